// dd4dvar.cu -- host side of the DD-4DVar library: geometry, workspace plan, the outer driver of
// Algorithm 1 and the C-ABI of include/dd4dvar.h.  All arithmetic of the
// hot path runs in the kernels of generic_kernels.cuh / fused_kernels.cuh / lbfgs_kernels.cuh /
// exchange_kernels.cuh; there is no CPU fallback.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <string>
#include <vector>

#include "../../include/dd4dvar.h"
#include "common.cuh"
#include "exchange_kernels.cuh"
#include "fused_kernels.cuh"
#include "generic_kernels.cuh"
#include "lbfgs_kernels.cuh"
#include "peaks_kernels.cuh"
#include "step_kernels.cuh"
#include "wave_forward.cuh"
#include "wave_adjoint.cuh"
#include "cost_kernels.cuh"
#include "gn_kernels.cuh"

namespace {

constexpr int NT_GK = 256;     // generic kernels: threads per block
constexpr int NT_RED = 256;    // cost reduction
constexpr int NT_LB = 512;     // L-BFGS CTA
#ifndef DD_EH_CHUNKS
#define DD_EH_CHUNKS 6
#endif
constexpr int EH_CHUNKS = DD_EH_CHUNKS;     // eval_local_host: chunks of subdomains whose copies overlap the sweeps of the others

struct Arena {
    char* base = nullptr;
    size_t off = 0, cap = 0;
    template <class T> T* take(size_t n)
    {
        off = (off + 255) & ~size_t(255);
        T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
        off += n * sizeof(T);
        return p;
    }
};

void* ar_take_bytes(void* arena, size_t bytes) { return static_cast<Arena*>(arena)->take<char>(bytes); }

// plan of the wavefront kernels (wave_common.cuh) for one layout
struct WavePlan {
    int enabled = 0, K = 3, grid = 0;
    int maxex = 0, maxey = 0, maxpx = 0, maxpy = 0;
    size_t smem_fwd = 0, smem_adj = 0;
    int* counter = nullptr;
    double* wtab = nullptr;             // [p2][maxpy + 2][8] row tables per tile row (wave_common.cuh)
    int wtab_stride = 0;
    double* lamW = nullptr;             // [ctot] adjoint variable at the window end (ck_cost -> wk_adjoint)
};

struct Layout {
    int p1 = 1, p2 = 1, q = 1, o = 0, nsub = 0;
    bool lbfgs = false;
    int path = 1;                       // 1 generic (block-tiled step kernels), 2 fused row-marching, 3 generic per-stage kernels, 4 wavefront
    int tiles_x = 1, ntiles = 1;        // 32x16 output tiles of the step kernels
    std::vector<Sub> hs;
    std::vector<NbRect> hnb;
    NbRect* dnb = nullptr;
    std::vector<int> colown, rowown, ncolcov, colcov, nrowcov, rowcov, tc_ei0, tc_ex, tr_ej0, tr_ey, wb;
    long long ctot = 0, ttot = 0, gtot = 0, ptot1 = 0, otot = 0, etot = 0, vtot = 0;
    int maxnovl = 0;
    double* ovl = nullptr;              // overlap store (option overlap_levels, generic path)
    int maxnpad = 0, maxncell = 0, maxnring = 0, Wmax = 0, CB = 1, maxcov = 1;
    // device
    Sub* dsubs = nullptr;
    GeoP geo{};
    int* itab = nullptr;
    double *x = nullptr, *xbs = nullptr, *xfrozen = nullptr, *pred_end = nullptr, *gx = nullptr;
    double *traj = nullptr, *ghost = nullptr, *gedge = nullptr;
    double *Zp = nullptr, *Za = nullptr, *lamA = nullptr, *lamB = nullptr, *A = nullptr;
    double *H1 = nullptr, *HB = nullptr, *P = nullptr, *UB = nullptr;
    double *partial = nullptr, *parts = nullptr, *Jev = nullptr, *dmax = nullptr;
    double *w = nullptr, *wt = nullptr, *g = nullptr, *gn = nullptr, *d = nullptr, *S = nullptr, *Y = nullptr;
    LbfgsState st{};
    int* okmask = nullptr;
    int* cmask = nullptr;
    int *own = nullptr, *notown = nullptr;  // sharded runs: 1 for the subdomains this process owns / does not own
    bool sharded = false;
    int own_j0 = 0, own_j1 = 0;               // [EH_CHUNKS][nsub] subdomain masks of the chunks of eval_local_host
    // observations binned per (subdomain, local level)
    bool have_obs = false;
    long long* obs_start = nullptr;
    int* obs_idx = nullptr;
    int* obs_lj = nullptr;
    double *obs_y = nullptr, *obs_c = nullptr, *obs_r = nullptr;
    double* obs_rt = nullptr;           // Gauss-Newton: forcing 2 c H dZ of the tangent-linear sweep
    double *gn_lamW = nullptr, *gn_gx = nullptr, *gn_Hp = nullptr;     // Gauss-Newton: [ctot] each
    double *gn_dtraj = nullptr, *gn_zero = nullptr;                    // Gauss-Newton on generic layouts: TLM trajectory [ttot], zeros
    FusedPlan fp{};
    WavePlan wp{};
};

}  // namespace

struct dd4dvar_s {
    dd4dvar_grid grid;
    dd4dvar_decomp dec;
    dd4dvar_window win;
    dd4dvar_opts opt;
    cudaStream_t stream = nullptr;
    std::string err;
    long long launches = 0;
    // model tables
    std::vector<double> h_tab;          // 6 x nlat
    std::vector<double> h_ctab;         // staging of the row-marching kernels' padded tables
    double* d_tab = nullptr;
    double* d_ctab = nullptr;           // [6][FK_CTAB], per handle
    ModelP mp{};
    CostP cp{};
    double sig_o[3] = { 1, 1, 1 };
    Layout G, L;
    bool have_ws = false, have_bg = false;
    int coop_grid = 0;                  // resident CTAs of sk_forward_multi (0: cooperative launch not available)
    bool overlap_levels = false;        // (25c) case 1 on every level of the window (generic path only)
    bool history_global = true;         // evaluate J of eq (6) at the gathered analysis after every outer iteration
    void* ws = nullptr;
    size_t ws_bytes = 0;
    // eval_local_host: copy streams and events (created on first use, destroyed with the handle)
    cudaStream_t s_h2d = nullptr, s_d2h = nullptr;
    cudaEvent_t ev_in = nullptr, ev_h2d[EH_CHUNKS] = {}, ev_sw[EH_CHUNKS] = {}, ev_out = nullptr;
    int* h_pin = nullptr;               // pinned scratch for small read-backs
    // dd4dvar_set_phase_timing: CUDA-event marks inside dd4dvar_run (off by default: no event is recorded)
    bool ph_on = false;
    std::vector<cudaEvent_t> ph_ev;     // pool, reused by every run
    std::vector<int> ph_kind;           // ph_kind[i] = phase that starts at mark i (-1: none)
    double ph_ms[5] = { 0, 0, 0, 0, 0 };
    std::vector<double> h_tmp;
};

namespace {

int fail(dd4dvar_t h, int code, const std::string& msg)
{
    if (h) h->err = msg;
    return code;
}
#define CU(call)                                                                         \
    do {                                                                                 \
        cudaError_t e_ = (call);                                                         \
        if (e_ != cudaSuccess)                                                           \
            return fail(h, -4, std::string(#call) + ": " + cudaGetErrorString(e_));      \
    } while (0)
#define LAUNCH(kern, grid, block, ...)                        \
    do {                                                      \
        kern<<<grid, block, 0, h->stream>>>(__VA_ARGS__);     \
        ++h->launches;                                        \
    } while (0)

int imod(int a, int n) { int r = a % n; return r < 0 ? r + n : r; }

// ---- geometry: Def 3 l.128-154, Def 16 l.755-763, eq (70) l.1024; ragged split DESIGN.md R9
int build_layout(Layout& L, int nlon, int nlat, int N, int p1, int p2, int q, int o)
{
    L.p1 = p1; L.p2 = p2; L.q = q; L.o = o;
    if (p1 < 1 || p2 < 1 || q < 1 || o < 0 || q > N) return -2;
    if ((long long)p1 * p2 * q > 65535) return -2;
    L.nsub = p1 * p2 * q;
    L.wb.resize(q + 1);
    for (int j = 0; j <= q; ++j) L.wb[j] = (int)(((long long)j * N) / q);
    L.tc_ei0.resize(p1); L.tc_ex.resize(p1); L.tr_ej0.resize(p2); L.tr_ey.resize(p2);
    std::vector<int> oi0(p1), oi1(p1), oj0(p2), oj1(p2), gys(p2), gyn(p2);
    for (int a = 0; a < p1; ++a) {
        oi0[a] = (int)(((long long)a * nlon) / p1); oi1[a] = (int)(((long long)(a + 1) * nlon) / p1);
        if (oi1[a] <= oi0[a]) return -2;
        if (p1 == 1) { L.tc_ei0[a] = 0; L.tc_ex[a] = nlon; }
        else { L.tc_ei0[a] = oi0[a] - o; L.tc_ex[a] = oi1[a] - oi0[a] + 2 * o; }
        if (L.tc_ex[a] > nlon) return -2;
    }
    for (int b = 0; b < p2; ++b) {
        oj0[b] = (int)(((long long)b * nlat) / p2); oj1[b] = (int)(((long long)(b + 1) * nlat) / p2);
        if (oj1[b] <= oj0[b]) return -2;
        int j0 = std::max(oj0[b] - o, 0), j1 = std::min(oj1[b] + o, nlat);
        L.tr_ej0[b] = j0; L.tr_ey[b] = j1 - j0;
        gys[b] = j0 == 0 ? 0 : DD_GHOST; gyn[b] = j1 == nlat ? 0 : DD_GHOST;
        if (j0 - gys[b] < 0 || j1 + gyn[b] > nlat) return -2;        // ghost ring off the grid
    }
    L.colown.assign(nlon, 0); L.rowown.assign(nlat, 0);
    L.ncolcov.assign(nlon, 0); L.colcov.assign(4 * nlon, 0);
    L.nrowcov.assign(nlat, 0); L.rowcov.assign(4 * nlat, 0);
    for (int a = 0; a < p1; ++a) {
        for (int i = oi0[a]; i < oi1[a]; ++i) L.colown[i] = a;
        for (int li = 0; li < L.tc_ex[a]; ++li) {
            int gi = imod(L.tc_ei0[a] + li, nlon);
            if (L.ncolcov[gi] >= 4) return -2;
            L.colcov[4 * gi + L.ncolcov[gi]++] = a;
        }
    }
    for (int b = 0; b < p2; ++b) {
        for (int j = oj0[b]; j < oj1[b]; ++j) L.rowown[j] = b;
        for (int lj = 0; lj < L.tr_ey[b]; ++lj) {
            int gj = L.tr_ej0[b] + lj;
            if (L.nrowcov[gj] >= 4) return -2;
            L.rowcov[4 * gj + L.nrowcov[gj]++] = b;
        }
    }
    int mc = 1, mr = 1;
    for (int v : L.ncolcov) mc = std::max(mc, v);
    for (int v : L.nrowcov) mr = std::max(mr, v);
    L.maxcov = mc * mr;
    L.hs.resize(L.nsub);
    L.ctot = L.ttot = L.gtot = L.ptot1 = L.otot = L.etot = L.vtot = 0; L.maxnovl = 0;
    L.maxnpad = L.maxncell = L.maxnring = L.Wmax = 0;
    for (int jw = 0; jw < q; ++jw)
        for (int b = 0; b < p2; ++b)
            for (int a = 0; a < p1; ++a) {
                Sub& s = L.hs[(jw * p2 + b) * p1 + a];
                s.a = a; s.b = b; s.jw = jw;
                s.oi0 = oi0[a]; s.oi1 = oi1[a]; s.oj0 = oj0[b]; s.oj1 = oj1[b];
                s.ei0 = L.tc_ei0[a]; s.ej0 = L.tr_ej0[b]; s.ex = L.tc_ex[a]; s.ey = L.tr_ey[b];
                s.gx = p1 == 1 ? 0 : DD_GHOST; s.gys = gys[b]; s.gyn = gyn[b];
                s.px = s.ex + 2 * s.gx; s.py = s.ey + s.gys + s.gyn;
                s.s = L.wb[jw]; s.W = L.wb[jw + 1] - L.wb[jw];
                if (s.W < 1) return -2;
                s.ncell = s.ex * s.ey; s.npad = s.px * s.py; s.nring = s.npad - s.ncell;
                s.coff = L.ctot; s.toff = L.ttot; s.goff = L.gtot; s.poff = 3 * L.ptot1; s.ooff = L.otot;
                s.eoff = L.etot; L.etot += (long long)s.W * 2 * s.py;
                // keep every plane 16-byte aligned relative to 256-byte aligned array bases
                L.ctot += 3LL * s.ncell; L.ctot = (L.ctot + 1) & ~1LL;
                L.ttot += (long long)(s.W + 1) * 3 * s.ncell; L.ttot = (L.ttot + 1) & ~1LL;
                L.gtot += (long long)s.W * 3 * s.nring; L.gtot = (L.gtot + 1) & ~1LL;
                L.ptot1 += s.npad;
                L.otot += s.W + 2;
                L.maxnpad = std::max(L.maxnpad, s.npad); L.maxncell = std::max(L.maxncell, s.ncell);
                L.maxnring = std::max(L.maxnring, s.nring); L.Wmax = std::max(L.Wmax, s.W);
            }
    // spatial-overlap rectangles of every subdomain with the other tiles of its window (periodic in longitude)
    L.hnb.clear();
    for (int k = 0; k < L.nsub; ++k) {
        Sub& s = L.hs[k];
        s.nb0 = (int)L.hnb.size(); s.novl = 0;
        for (int b2 = 0; b2 < p2; ++b2)
            for (int a2 = 0; a2 < p1; ++a2) {
                if (a2 == s.a && b2 == s.b) continue;
                const Sub& t = L.hs[(s.jw * p2 + b2) * p1 + a2];
                const int j0 = std::max(s.ej0, t.ej0), j1 = std::min(s.ej0 + s.ey, t.ej0 + t.ey);
                if (j1 <= j0) continue;
                for (int sh = -1; sh <= 1; ++sh) {
                    const int t0 = t.ei0 + sh * nlon;
                    const int i0 = std::max(s.ei0, t0), i1 = std::min(s.ei0 + s.ex, t0 + t.ex);
                    if (i1 <= i0) continue;
                    NbRect r;
                    r.coff2 = t.coff; r.toff2 = t.toff; r.ex2 = t.ex; r.ncell2 = t.ncell;
                    r.ooff = s.novl; s.novl += (i1 - i0) * (j1 - j0);
                    r.i0 = i0 - s.ei0; r.j0 = j0 - s.ej0; r.w = i1 - i0; r.h = j1 - j0;
                    r.ni0 = i0 - t0; r.nj0 = j0 - t.ej0;
                    L.hnb.push_back(r);
                }
            }
        s.nnb = (int)L.hnb.size() - s.nb0;
        s.voff = L.vtot; L.vtot += (long long)s.W * 3 * s.novl;
        L.maxnovl = std::max(L.maxnovl, s.novl);
    }
    {
        int mex = 0, mey = 0;
        for (const Sub& q : L.hs) { mex = std::max(mex, q.ex); mey = std::max(mey, q.ey); }
        L.tiles_x = (mex + SK_TX - 1) / SK_TX; L.ntiles = L.tiles_x * ((mey + SK_TY - 1) / SK_TY);
    }
    L.CB = std::min(64, std::max(1, (3 * L.maxncell + NT_RED * 32 - 1) / (NT_RED * 32)));
    return 0;
}

// device arrays of one layout, taken from the arena in a fixed order (dry run = size query)
void plan_layout(Layout& L, Arena& ar, int nlon, int nlat, int m)
{
    L.dsubs = ar.take<Sub>(L.nsub);
    L.dnb = ar.take<NbRect>(L.hnb.size() + 1);
    const size_t nit = (size_t)nlon * 6 + (size_t)nlat * 6 + 2 * L.p1 + 2 * L.p2 + L.q + 1;
    L.itab = ar.take<int>(nit);
    L.x = ar.take<double>(L.ctot); L.xbs = ar.take<double>(L.ctot); L.gx = ar.take<double>(L.ctot);
    L.xfrozen = ar.take<double>(L.ctot); L.pred_end = ar.take<double>(L.ctot);
    L.traj = ar.take<double>(L.ttot);
    L.ghost = ar.take<double>(std::max<long long>(L.gtot, 2));
    L.Zp = ar.take<double>(3 * L.ptot1); L.Za = ar.take<double>(3 * L.ptot1);
    L.lamA = ar.take<double>(3 * L.ptot1); L.lamB = ar.take<double>(3 * L.ptot1);
    L.A = ar.take<double>(3 * L.ptot1);
    L.H1 = ar.take<double>(L.ptot1); L.HB = ar.take<double>(L.ptot1);
    L.P = ar.take<double>(L.ptot1); L.UB = ar.take<double>(L.ptot1);
    L.partial = ar.take<double>((size_t)L.nsub * L.CB * 5);
    L.parts = ar.take<double>((size_t)L.nsub * 5);
    L.Jev = ar.take<double>(L.nsub);
    L.dmax = ar.take<double>(L.nsub);
    L.okmask = ar.take<int>(L.nsub);
    L.cmask = ar.take<int>((size_t)EH_CHUNKS * L.nsub);
    L.own = ar.take<int>(L.nsub); L.notown = ar.take<int>(L.nsub);
    if (L.lbfgs) {
        L.w = ar.take<double>(L.ctot); L.wt = ar.take<double>(L.ctot); L.g = ar.take<double>(L.ctot);
        L.gn = ar.take<double>(L.ctot); L.d = ar.take<double>(L.ctot);
        L.S = ar.take<double>((size_t)std::max(m, 1) * L.ctot); L.Y = ar.take<double>((size_t)std::max(m, 1) * L.ctot);
        L.st.J = ar.take<double>(L.nsub); L.st.Jt = ar.take<double>(L.nsub); L.st.t = ar.take<double>(L.nsub);
        L.st.gd = ar.take<double>(L.nsub);
        L.st.nh = ar.take<int>(L.nsub); L.st.head = ar.take<int>(L.nsub); L.st.active = ar.take<int>(L.nsub);
        L.st.ok = ar.take<int>(L.nsub); L.st.done = ar.take<int>(L.nsub); L.st.trial = ar.take<int>(L.nsub);
        L.st.rho = ar.take<double>((size_t)L.nsub * std::max(m, 1));
        L.st.gam = ar.take<double>((size_t)L.nsub * std::max(m, 1));
        L.st.nactive = ar.take<int>(4);
    }
    if ((L.path == 1 || L.path == 3) && L.vtot > 0) L.ovl = ar.take<double>(L.vtot);
    if ((L.path == 1 || L.path == 3) && L.lbfgs) {
        L.gn_gx = ar.take<double>(L.ctot); L.gn_Hp = ar.take<double>(L.ctot);
        L.gn_dtraj = ar.take<double>(L.ttot);
        L.gn_zero = ar.take<double>(std::max(L.ctot, L.vtot) + 2);
    }
    fused_plan_arrays(L.fp, ar_take_bytes, &ar);
    if (L.wp.enabled) {
        L.gedge = ar.take<double>(std::max<long long>(L.etot, 2));
        L.wp.counter = ar.take<int>(16);
        L.wp.wtab_stride = (L.wp.maxpy + 2) * 8;
        L.wp.wtab = ar.take<double>((size_t)L.p2 * L.wp.wtab_stride);
        L.wp.lamW = ar.take<double>(L.ctot);
        if (L.lbfgs) { L.gn_lamW = ar.take<double>(L.ctot); L.gn_gx = ar.take<double>(L.ctot); L.gn_Hp = ar.take<double>(L.ctot); }
    }
}

// eligibility and shared-memory budget of the wavefront kernels (wave_common.cuh)
void wave_plan_init(WavePlan& wp, const Sub* subs, int nsub)
{
    wp = WavePlan();
    if (!subs || nsub <= 0) return;
    for (int k = 0; k < nsub; ++k) {
        const Sub& s = subs[k];
        if (s.gx != DD_GHOST || (s.ex & 1) || s.ey > 1000 || s.ex < 2 || s.ex > 255) return;
        if ((s.gys != 0 && s.gys != DD_GHOST) || (s.gyn != 0 && s.gyn != DD_GHOST)) return;
        if (s.W < 4) return;            // WK_NTAB row-table slots cover the steps in flight only if every window has >= 4 steps
        wp.maxex = std::max(wp.maxex, s.ex); wp.maxey = std::max(wp.maxey, s.ey);
        wp.maxpx = std::max(wp.maxpx, s.px); wp.maxpy = std::max(wp.maxpy, s.py);
    }
    if (wp.maxpx - 4 <= 64) wp.K = 2;
    else if (wp.maxpx - 4 <= 96) wp.K = 3;
    else return;
    if (wp.maxey > WK_AROWS(wp.K)) return;      // rows of the adjoint kernel's resident state (compile-time field stride)
    wp.smem_fwd = sizeof(double) * (size_t)wk_layout(false, wp.maxex, wp.maxey, wp.maxpx, wp.maxpy).total;
    wp.smem_adj = sizeof(double) * (size_t)wk_layout(true, wp.maxex, wp.maxey, wp.maxpx, wp.maxpy).total;
    if (wp.smem_fwd > WK_SMEM_MAX || wp.smem_adj > WK_SMEM_MAX) return;
    wp.enabled = 1;
}

// eval_local_host: bounds of its EH_CHUNKS chunks of consecutive subdomains.  A CTA of the wavefront kernels takes the
// subdomains k = b, b + grid, ... in turn (wave_common.cuh), so there the bounds are multiples of the grid size: every
// chunk is a whole number of rounds and the masked sweeps together take as many rounds as one full sweep.  A round is
// copied in (or out) in about half the time it is swept, so the copy of a chunk hides behind the sweep of a neighbour of
// half its size: chunks of 1, 2, .. rounds from either end (what is exposed is the first round's copy in and the last
// round's copy out), the two in the middle share the rest (config 3: 14 rounds = 1 + 2 + 4 + 4 + 2 + 1).
void eh_bounds(const Layout& L, int* kb)
{
    const int gran = L.wp.enabled && L.wp.grid > 0 ? L.wp.grid : 0;
    const int R = gran ? (L.nsub + gran - 1) / gran : 0;
    constexpr int NE = (EH_CHUNKS - 2) / 2;             // doubling chunks at either end
    if (EH_CHUNKS >= 4 && EH_CHUNKS % 2 == 0 && R >= 4 * ((1 << NE) - 1) + 2) {
        int r[EH_CHUNKS];
        int used = 0;
        for (int i = 0; i < NE; ++i) { r[i] = r[EH_CHUNKS - 1 - i] = 1 << i; used += 2 << i; }
        r[NE] = (R - used + 1) / 2; r[NE + 1] = (R - used) / 2;
        kb[0] = 0;
        for (int c = 0; c < EH_CHUNKS; ++c) kb[c + 1] = std::min(L.nsub, kb[c] + gran * r[c]);
        kb[EH_CHUNKS] = L.nsub;
        return;
    }
    for (int c = 0; c <= EH_CHUNKS; ++c) {
        const long long k = ((long long)c * L.nsub + EH_CHUNKS - 1) / EH_CHUNKS;
        kb[c] = k > L.nsub ? L.nsub : (int)k;
    }
}

int upload_chunk_masks(dd4dvar_t h, Layout& L)
{
    int kb[EH_CHUNKS + 1];
    eh_bounds(L, kb);
    std::vector<int> cm((size_t)EH_CHUNKS * L.nsub, 0);
    for (int c = 0; c < EH_CHUNKS; ++c)
        for (int k = kb[c]; k < kb[c + 1]; ++k) cm[(size_t)c * L.nsub + k] = 1;
    CU(cudaMemcpyAsync(L.cmask, cm.data(), sizeof(int) * cm.size(), cudaMemcpyHostToDevice, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    return 0;
}

int upload_layout(dd4dvar_t h, Layout& L)
{
    const int nlon = h->grid.nlon, nlat = h->grid.nlat;
    CU(cudaMemcpyAsync(L.dsubs, L.hs.data(), sizeof(Sub) * L.nsub, cudaMemcpyHostToDevice, h->stream));
    if (!L.hnb.empty())
        CU(cudaMemcpyAsync(L.dnb, L.hnb.data(), sizeof(NbRect) * L.hnb.size(), cudaMemcpyHostToDevice, h->stream));
    std::vector<int> t;
    auto put = [&](const std::vector<int>& v) { size_t o = t.size(); t.insert(t.end(), v.begin(), v.end()); return o; };
    const size_t o_colown = put(L.colown), o_ncolcov = put(L.ncolcov), o_colcov = put(L.colcov);
    const size_t o_rowown = put(L.rowown), o_nrowcov = put(L.nrowcov), o_rowcov = put(L.rowcov);
    const size_t o_ei0 = put(L.tc_ei0), o_ex = put(L.tc_ex), o_ej0 = put(L.tr_ej0), o_ey = put(L.tr_ey);
    const size_t o_wb = put(L.wb);
    CU(cudaMemcpyAsync(L.itab, t.data(), sizeof(int) * t.size(), cudaMemcpyHostToDevice, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    GeoP& g = L.geo;
    g.nlon = nlon; g.nlat = nlat; g.p1 = L.p1; g.p2 = L.p2; g.q = L.q;
    g.colown = L.itab + o_colown; g.ncolcov = L.itab + o_ncolcov; g.colcov = L.itab + o_colcov;
    g.rowown = L.itab + o_rowown; g.nrowcov = L.itab + o_nrowcov; g.rowcov = L.itab + o_rowcov;
    g.tc_ei0 = L.itab + o_ei0; g.tc_ex = L.itab + o_ex; g.tr_ej0 = L.itab + o_ej0; g.tr_ey = L.itab + o_ey;
    g.wb = L.itab + o_wb;
    // adjoint buffers: the ghost ring must be (and stays) zero
    CU(cudaMemsetAsync(L.lamA, 0, sizeof(double) * 3 * L.ptot1, h->stream));
    CU(cudaMemsetAsync(L.lamB, 0, sizeof(double) * 3 * L.ptot1, h->stream));
    if (L.gn_zero) CU(cudaMemsetAsync(L.gn_zero, 0, sizeof(double) * (std::max(L.ctot, L.vtot) + 2), h->stream));
    CU(cudaMemsetAsync(L.xfrozen, 0, sizeof(double) * L.ctot, h->stream));
    CU(cudaMemsetAsync(L.pred_end, 0, sizeof(double) * L.ctot, h->stream));
    CU(cudaMemsetAsync(L.x, 0, sizeof(double) * L.ctot, h->stream));
    CU(cudaMemsetAsync(L.xbs, 0, sizeof(double) * L.ctot, h->stream));
    if (L.lbfgs) {
        CU(cudaMemsetAsync(L.w, 0, sizeof(double) * L.ctot, h->stream));
        CU(cudaMemsetAsync(L.st.nh, 0, sizeof(int) * L.nsub, h->stream));
        CU(cudaMemsetAsync(L.st.head, 0, sizeof(int) * L.nsub, h->stream));
        CU(cudaMemsetAsync(L.st.done, 0, sizeof(int) * L.nsub, h->stream));
    }
    return 0;
}

// ---- sweeps (generic path) -------------------------------------------------------------
dim3 pad_grid(const Layout& L) { return dim3((L.maxnpad + NT_GK - 1) / NT_GK, L.nsub); }
dim3 cell_grid(const Layout& L) { return dim3((L.maxncell + NT_GK - 1) / NT_GK, L.nsub); }

void forward_generic(dd4dvar_t h, Layout& L, const int* mask)
{
    // level 0 of the store = the control
    LAUNCH(gk_store_control, cell_grid(L), NT_GK, L.dsubs, mask, L.x, L.traj);
    if (L.path != 3) {
        if (h->coop_grid > 0 && L.Wmax > 1) {
            // all steps in one cooperative launch (grid-wide barrier between the steps)
            const Sub* subs = L.dsubs; int n0 = 0, n1 = L.Wmax, tiles_x = L.tiles_x, ntiles = L.ntiles, nsub = L.nsub;
            double* traj = L.traj; const double* ghost = L.ghost; ModelP mp = h->mp;
            void* args[] = { &subs, &mask, &n0, &n1, &mp, &traj, &ghost, &tiles_x, &ntiles, &nsub };
            const int grid = std::min(h->coop_grid, L.ntiles * L.nsub);
            if (cudaLaunchCooperativeKernel((const void*)sk_forward_multi, dim3(grid), dim3(SK_NT), args, 0, h->stream) == cudaSuccess) {
                ++h->launches;
                return;
            }
            cudaGetLastError();                 // fall back to one launch per step
        }
        for (int n = 0; n < L.Wmax; ++n)
            LAUNCH(sk_forward_step, dim3(L.ntiles, L.nsub), SK_NT, L.dsubs, mask, n, h->mp, L.traj, L.ghost, L.tiles_x);
        return;
    }
    for (int n = 0; n < L.Wmax; ++n) {
        LAUNCH(gk_fill_pad, pad_grid(L), NT_GK, L.dsubs, mask, n, L.traj, L.ghost, L.Zp);
        LAUNCH(gk_stageA, pad_grid(L), NT_GK, L.dsubs, mask, n, h->mp, L.Zp, L.Za);
        LAUNCH(gk_stageH, pad_grid(L), NT_GK, L.dsubs, mask, n, h->mp, L.Za, L.H1);
        LAUNCH(gk_stageUV, pad_grid(L), NT_GK, L.dsubs, mask, n, h->mp, L.Za, L.H1, L.traj);
    }
}
void cost_generic(dd4dvar_t h, Layout& L, const int* mask, double* Jout)
{
    LAUNCH(gk_cost_partial<NT_RED>, dim3(L.CB, L.nsub), NT_RED, L.dsubs, mask, L.geo, h->cp, L.x, L.xbs,
           L.xfrozen, L.pred_end, L.traj, L.have_obs ? L.obs_start : nullptr, L.obs_idx, L.obs_y, L.obs_c,
           L.partial);
    LAUNCH(gk_cost_final, (L.nsub + 127) / 128, 128, L.nsub, mask, L.CB, L.partial, L.parts, Jout);
    if (h->overlap_levels && L.ovl)
        LAUNCH(gk_ovl_cost<NT_RED>, L.nsub, NT_RED, L.dsubs, L.dnb, mask, h->cp, L.traj, L.ovl, L.parts, Jout);
}
// lin != nullptr: the same sweep as the adjoint of the TANGENT-LINEAR misfits (Gauss-Newton product, gn_kernels.cuh): the
// forcing terms are taken from the tangent-linear trajectory `lin` against zeros (they are linear in it), the control-level
// terms from the perturbation dx; the step adjoints still linearise about L.traj.
void adjoint_generic(dd4dvar_t h, Layout& L, const int* mask, double* gw, const double* lin = nullptr,
                     const double* dx = nullptr, const double* zero = nullptr, const double* zero_obs = nullptr,
                     double* gx_out = nullptr)
{
    double* buf[2] = { L.lamA, L.lamB };
    const double* ftraj = lin ? lin : L.traj;
    const double* fxf = lin ? zero : L.xfrozen;
    LAUNCH(gk_adj_init, cell_grid(L), NT_GK, L.dsubs, mask, L.Wmax, L.q, L.p1 * L.p2, h->cp, ftraj,
           fxf, L.lamA, L.lamB);
    for (int n = L.Wmax; n >= 0; --n) {
        double* cur = buf[(L.Wmax - n) & 1];
        double* nxt = buf[(L.Wmax - n + 1) & 1];
        if (L.have_obs)
            LAUNCH(gk_obs_force, dim3(4, L.nsub), NT_GK, L.dsubs, mask, n, L.obs_start, L.obs_idx, lin ? zero_obs : L.obs_y,
                   L.obs_c, ftraj, cur);
        if (n > 0 && h->overlap_levels && L.ovl)
            LAUNCH(gk_ovl_force, cell_grid(L), NT_GK, L.dsubs, L.dnb, mask, n, h->cp, ftraj, lin ? zero : L.ovl, cur);
        if (n > 0 && L.path != 3) {
            sk_adjoint_step<<<dim3(L.ntiles, L.nsub), SK_NT, sizeof(double) * SK_ADJ_SMEM_DOUBLES, h->stream>>>(
                L.dsubs, mask, n - 1, h->mp, L.traj, L.ghost, cur, nxt, L.tiles_x);
            ++h->launches;
        } else if (n > 0) {
            LAUNCH(gk_fill_pad, pad_grid(L), NT_GK, L.dsubs, mask, n - 1, L.traj, L.ghost, L.Zp);
            LAUNCH(gk_stageA, pad_grid(L), NT_GK, L.dsubs, mask, n - 1, h->mp, L.Zp, L.Za);
            LAUNCH(gk_adjHB, pad_grid(L), NT_GK, L.dsubs, mask, n - 1, h->mp, L.Za, cur, L.traj, L.HB, L.P, L.UB);
            LAUNCH(gk_adjA, pad_grid(L), NT_GK, L.dsubs, mask, n - 1, h->mp, L.Za, cur, L.HB, L.P, L.UB, L.A);
            LAUNCH(gk_adjL0, pad_grid(L), NT_GK, L.dsubs, mask, n - 1, h->mp, L.Zp, L.A, nxt);
        }
    }
    if (lin)
        LAUNCH(gk_grad_final, cell_grid(L), NT_GK, L.dsubs, mask, L.geo, h->cp, dx, zero, zero, zero, buf[L.Wmax & 1],
               gx_out, gw);
    else
        LAUNCH(gk_grad_final, cell_grid(L), NT_GK, L.dsubs, mask, L.geo, h->cp, L.x, L.xbs, L.xfrozen,
               L.pred_end, buf[L.Wmax & 1], L.gx, gw);
}


WkArgs wave_args(dd4dvar_t h, Layout& L, const int* mask, double* Jout, double* gw)
{
    WkArgs a;
    a.subs = L.dsubs; a.nbr = L.dnb; a.mask = mask; a.nsub = L.nsub; a.counter = L.wp.counter;
    a.m = h->mp; a.cp = h->cp; a.geo = L.geo;
    a.x = L.x; a.xbs = L.xbs; a.xfrozen = L.xfrozen; a.pred_end = L.pred_end;
    a.traj = L.traj; a.ghost = L.ghost; a.gedge = L.gedge;
    a.obs_start = L.have_obs ? L.obs_start : nullptr; a.obs_idx = L.obs_idx; a.obs_lj = L.obs_lj;
    a.obs_y = L.obs_y; a.obs_c = L.obs_c; a.obs_r = L.obs_r;
    a.parts = L.parts; a.J = Jout; a.gx = L.gx; a.gw = gw;
    a.maxex = L.wp.maxex; a.maxey = L.wp.maxey; a.maxpx = L.wp.maxpx; a.maxpy = L.wp.maxpy;
    a.wtab = L.wp.wtab; a.wtab_stride = L.wp.wtab_stride; a.lamW = L.wp.lamW;
    a.Lf = wk_layout(false, a.maxex, a.maxey, a.maxpx, a.maxpy);
    a.La = wk_layout(true, a.maxex, a.maxey, a.maxpx, a.maxpy);
    return a;
}

// one evaluation of J_ji (and its gradient) on every (unmasked) subdomain: steps a1-a4
void adjoint_only(dd4dvar_t h, Layout& L, const int* mask, double* gw)
{
    if (L.path == 5) {
        // (consumes the control-level part of the gradient that ck_cost left in gx: one adjoint sweep per forward sweep)
        WkArgs a = wave_args(h, L, mask, nullptr, gw);
        if (L.wp.K == 2) wk_adjoint<2><<<L.wp.grid, WK_NT, L.wp.smem_adj, h->stream>>>(a);
        else wk_adjoint<3><<<L.wp.grid, WK_NT, L.wp.smem_adj, h->stream>>>(a);
        ++h->launches;
        if (gw) LAUNCH(ck_scale_grad, dim3(std::min(32, (3 * L.maxncell + 255) / 256), L.nsub), 256, L.dsubs, mask, h->cp, L.gx, gw);
        return;
    }
    if (L.path == 2 || L.path == 4) {
        {
            cudaMemsetAsync(L.fp.counter, 0, sizeof(int), h->stream);
            if (L.fp.nt == 64) fk64::fk_adjoint2<<<L.fp.nslots, 64, 0, h->stream>>>(
                L.dsubs, mask, h->mp, h->cp, L.geo, L.x, L.xbs, L.xfrozen, L.pred_end, L.traj, L.ghost,
                L.have_obs ? L.obs_start : nullptr, L.obs_idx, L.obs_y, L.obs_c, L.gx, gw, L.nsub, L.fp.scratch,
                L.fp.slot_stride, L.fp.counter, h->d_ctab);
            else fk128::fk_adjoint2<<<L.fp.nslots, 128, 0, h->stream>>>(
                L.dsubs, mask, h->mp, h->cp, L.geo, L.x, L.xbs, L.xfrozen, L.pred_end, L.traj, L.ghost,
                L.have_obs ? L.obs_start : nullptr, L.obs_idx, L.obs_y, L.obs_c, L.gx, gw, L.nsub, L.fp.scratch,
                L.fp.slot_stride, L.fp.counter, h->d_ctab);
        }
        ++h->launches;
        return;
    }
    adjoint_generic(h, L, mask, gw);
}
void sweep(dd4dvar_t h, Layout& L, bool with_adjoint, const int* mask, double* Jout, double* gw)
{
    if (L.path == 4 || L.path == 5) {
        // forward sweep + trajectory store + H (25b) in the wavefront kernel, then the control-level terms (ck_cost)
        WkArgs a = wave_args(h, L, mask, Jout, gw);
        if (L.wp.K == 2) wk_forward<2><<<L.wp.grid, WK_NT, L.wp.smem_fwd, h->stream>>>(a);
        else wk_forward<3><<<L.wp.grid, WK_NT, L.wp.smem_fwd, h->stream>>>(a);
        ++h->launches;
        ck_cost<<<L.nsub, CK_NT, 0, h->stream>>>(a);
        ++h->launches;
        if (with_adjoint) adjoint_only(h, L, mask, gw);
        return;
    }
    if (L.path == 2) {
        cudaMemsetAsync(L.fp.counter, 0, sizeof(int), h->stream);
        if (L.fp.nt == 64) fk64::fk_forward2<<<L.fp.nslots_fwd, 64, 0, h->stream>>>(L.dsubs, mask, h->mp, L.x, L.traj, L.ghost,
                                                                      L.nsub, L.fp.scratch, L.fp.slot_stride, L.fp.counter, h->d_ctab);
        else fk128::fk_forward2<<<L.fp.nslots_fwd, 128, 0, h->stream>>>(L.dsubs, mask, h->mp, L.x, L.traj, L.ghost,
                                                                      L.nsub, L.fp.scratch, L.fp.slot_stride, L.fp.counter, h->d_ctab);
        ++h->launches;
    } else forward_generic(h, L, mask);
    cost_generic(h, L, mask, Jout);
    if (with_adjoint) adjoint_only(h, L, mask, gw);
}

// Alg 1 l.465: this iteration's results become the next one's frozen data
void exchange(dd4dvar_t h, Layout& L)
{
    LAUNCH(xk_freeze<NT_RED>, L.nsub, NT_RED, L.dsubs, L.geo, L.traj, L.x, L.xfrozen, L.pred_end, L.dmax,
           L.sharded ? (const int*)L.own : (const int*)nullptr);
    if (L.maxnring > 0)
        LAUNCH(xk_ghost_fill, dim3((L.maxnring + 127) / 128, L.nsub, std::min(L.Wmax, 8)), 128, L.dsubs, L.geo,
               L.traj, L.ghost);
    if (h->overlap_levels && L.ovl && L.maxnovl > 0)
        LAUNCH(xk_ovl_fill, dim3((L.maxnovl + 127) / 128, L.nsub, std::min(L.Wmax, 8)), 128, L.dsubs, L.dnb, L.traj, L.ovl);
    if (L.wp.enabled)
        LAUNCH(xk_edge_ua, dim3((2 * L.wp.maxpy + 63) / 64, L.nsub, std::min(L.Wmax, 8)), 64, L.dsubs, h->mp,
               L.ghost, L.gedge);
}

int sync_check(dd4dvar_t h)
{
    CU(cudaStreamSynchronize(h->stream));
    CU(cudaGetLastError());
    return 0;
}

// Phase marks of dd4dvar_run (dd4dvar_set_phase_timing): a mark closes the phase that is open and opens phase `kind`
// (0 sweeps, 1 L-BFGS kernels and their host round trips, 2 exchange, 3 J_global diagnostic, 4 gather / other; -1 none).
enum { PH_SWEEP = 0, PH_LBFGS = 1, PH_EXCH = 2, PH_JGLOBAL = 3, PH_OTHER = 4 };
void ph_mark(dd4dvar_t h, int kind)
{
    if (!h->ph_on) return;
    const size_t i = h->ph_kind.size();
    if (i == h->ph_ev.size()) {
        cudaEvent_t e;
        if (cudaEventCreate(&e) != cudaSuccess) { h->ph_on = false; return; }
        h->ph_ev.push_back(e);
    }
    cudaEventRecord(h->ph_ev[i], h->stream);
    h->ph_kind.push_back(kind);
}
// after the stream has been synchronised: add the time between consecutive marks to the phase the first one opened
void ph_collect(dd4dvar_t h)
{
    if (!h->ph_on) return;
    for (size_t i = 0; i + 1 < h->ph_kind.size(); ++i) {
        float ms = 0.f;
        if (h->ph_kind[i] >= 0 && cudaEventElapsedTime(&ms, h->ph_ev[i], h->ph_ev[i + 1]) == cudaSuccess)
            h->ph_ms[h->ph_kind[i]] += ms;
    }
    h->ph_kind.clear();
}

// J of eq (6) at a global state already in G.x
int global_cost(dd4dvar_t h, double* out)
{
    sweep(h, h->G, false, nullptr, h->G.Jev, nullptr);
    CU(cudaMemcpyAsync(out, h->G.Jev, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    return sync_check(h);
}

size_t plan_all(dd4dvar_t h, char* base)
{
    Arena ar; ar.base = base;
    h->d_tab = ar.take<double>(6 * (size_t)h->grid.nlat);
    h->d_ctab = ar.take<double>(6 * (size_t)FK_CTAB);
    plan_layout(h->G, ar, h->grid.nlon, h->grid.nlat, h->opt.lbfgs_m);
    plan_layout(h->L, ar, h->grid.nlon, h->grid.nlat, h->opt.lbfgs_m);
    return ar.off + 256;
}

}  // namespace

// =============================================================================== C-ABI ====
extern "C" {

int dd4dvar_create(const dd4dvar_grid* grid, const dd4dvar_decomp* decomp, const dd4dvar_window* window,
                   const dd4dvar_opts* opts, void* cuda_stream, dd4dvar_t* out)
{
    if (!grid || !decomp || !window || !out) return -1;
    *out = nullptr;
    if (grid->nlon < 3 || grid->nlat < 2 || window->nsteps < 1 || !(grid->radius > 0)) return -1;
    dd4dvar_s* h = new dd4dvar_s();
    h->grid = *grid; h->dec = *decomp; h->win = *window;
    if (opts) h->opt = *opts;
    else { h->opt.lbfgs_m = 5; h->opt.n_inner = 5; h->opt.max_backtrack = 20; h->opt.armijo_c1 = 1e-4; h->opt.path = 0; }
    if (h->opt.lbfgs_m < 0 || h->opt.lbfgs_m > 32 || h->opt.n_inner < 0 || h->opt.max_backtrack < 0) { delete h; return -1; }
    h->stream = (cudaStream_t)cuda_stream;
    const int nlon = grid->nlon, nlat = grid->nlat;
    // O1 row tables (eq (60)-(62) l.945-954; cell-centred rows R2; clamped metric R3), dt folded in
    const double PI = 3.14159265358979323846;
    const double dlam = 2.0 * PI / nlon, dth = PI / nlat, dt = window->dt, a = grid->radius;
    std::vector<double> mc(nlat);
    h->h_tab.assign(6 * (size_t)nlat, 0.0);
    double* dtcz = &h->h_tab[0]; double* gdtcz = &h->h_tab[nlat]; double* dtf = &h->h_tab[2 * nlat];
    double* dtt = &h->h_tab[3 * nlat]; double* rp = &h->h_tab[4 * nlat]; double* rm = &h->h_tab[5 * nlat];
    for (int j = 0; j < nlat; ++j) {
        const double th = -0.5 * PI + (j + 0.5) * dth, c = cos(th);
        mc[j] = c > grid->cos_clamp ? c : grid->cos_clamp;
        const double cz = 1.0 / (2.0 * a * dlam * mc[j]);
        dtcz[j] = dt * cz; gdtcz[j] = grid->gravity * dt * cz;
        dtf[j] = dt * 2.0 * grid->omega * sin(th);
        dtt[j] = dt * sin(th) / (a * mc[j]);
    }
    for (int j = 0; j < nlat; ++j) {
        rp[j] = (j + 1 < nlat ? mc[j + 1] : mc[j]) / mc[j];
        rm[j] = (j > 0 ? mc[j - 1] : mc[j]) / mc[j];
    }
    const double cm = 1.0 / (2.0 * a * dth);
    h->mp.nlon = nlon; h->mp.nlat = nlat; h->mp.kap = grid->diffusion;
    h->mp.dtcm = dt * cm; h->mp.gdtcm = grid->gravity * dt * cm;
    h->cp.mu = decomp->mu; h->cp.lambda = decomp->lambda; h->cp.bgw = 0.0;
    for (int f = 0; f < 3; ++f) { h->cp.ib[f] = 1.0; h->cp.sb[f] = 1.0; }
    int rc = build_layout(h->G, nlon, nlat, window->nsteps, 1, 1, 1, 0);
    if (!rc) rc = build_layout(h->L, nlon, nlat, window->nsteps, decomp->p_lon, decomp->p_lat, decomp->q_time,
                               decomp->overlap);
    if (rc) { delete h; return rc; }
    h->G.lbfgs = false; h->L.lbfgs = true;
    h->G.path = 1;
    const bool fits = fused_fits(h->L.hs.data(), h->L.nsub) && nlat + 2 <= FK_CTAB;
    wave_plan_init(h->L.wp, h->L.hs.data(), h->L.nsub);
    const bool wave = h->L.wp.enabled && fits;
    if (h->opt.path == 2 && !fits) { delete h; return -2; }
    if ((h->opt.path == 4 || h->opt.path == 5) && !wave) { delete h; return -2; }
    if (h->opt.path < 0 || h->opt.path > 5) { delete h; return -1; }
    if (h->opt.path == 0) h->L.path = wave ? 5 : (fits ? 2 : 1);
    else h->L.path = h->opt.path;
    if (h->L.path != 4 && h->L.path != 5) h->L.wp = WavePlan();
    fused_plan_init(h->G.fp, nullptr, 0, 0);
    fused_plan_init(h->L.fp, (h->L.path == 2 || h->L.path == 4) ? h->L.hs.data() : nullptr, h->L.nsub, 0);
    h->ws_bytes = plan_all(h, nullptr);
    *out = h;
    return 0;
}

size_t dd4dvar_workspace_bytes(dd4dvar_t h) { return h ? h->ws_bytes : 0; }

int dd4dvar_set_workspace(dd4dvar_t h, void* d_buf, size_t bytes)
{
    if (!h || !d_buf) return fail(h, -1, "set_workspace: null argument");
    if (bytes < h->ws_bytes) return fail(h, -1, "set_workspace: buffer smaller than dd4dvar_workspace_bytes");
    if (((uintptr_t)d_buf & 255) != 0) return fail(h, -1, "set_workspace: buffer not 256-byte aligned");
    int ndev = 0;
    CU(cudaGetDeviceCount(&ndev));
    h->ws = d_buf;
    plan_all(h, (char*)d_buf);
    const int nlat = h->grid.nlat;
    CU(cudaMemcpyAsync(h->d_tab, h->h_tab.data(), sizeof(double) * 6 * nlat, cudaMemcpyHostToDevice, h->stream));
    h->mp.dtcz = h->d_tab; h->mp.gdtcz = h->d_tab + nlat; h->mp.dtf = h->d_tab + 2 * nlat;
    h->mp.dtt = h->d_tab + 3 * nlat; h->mp.rp = h->d_tab + 4 * nlat; h->mp.rm = h->d_tab + 5 * nlat;
    int rc = upload_layout(h, h->G);
    if (rc) return rc;
    rc = upload_layout(h, h->L);
    if (rc) return rc;
    if (cudaFuncSetAttribute(sk_adjoint_step, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)(sizeof(double) * SK_ADJ_SMEM_DOUBLES)) != cudaSuccess)
        return fail(h, -4, "shared-memory opt-in of sk_adjoint_step failed");
    {
        int dev = 0, nsm = 0, coop = 0, per_sm = 0;
        CU(cudaGetDevice(&dev));
        CU(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
        CU(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
        if (coop && cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, sk_forward_multi, SK_NT, 0) == cudaSuccess)
            h->coop_grid = per_sm * nsm;
    }
    if (cudaFuncSetAttribute(tk_step, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)(sizeof(double) * TK_SMEM_DOUBLES)) != cudaSuccess)
        return fail(h, -4, "shared-memory opt-in of tk_step failed");
    if (h->L.wp.enabled) {
        int dev = 0, nsm = 0;
        CU(cudaGetDevice(&dev));
        CU(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
        h->L.wp.grid = std::max(1, std::min(nsm, h->L.nsub));
        cudaError_t e1 = h->L.wp.K == 2
            ? cudaFuncSetAttribute(wk_forward<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->L.wp.smem_fwd)
            : cudaFuncSetAttribute(wk_forward<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->L.wp.smem_fwd);
        cudaError_t e2 = h->L.wp.K == 2
            ? cudaFuncSetAttribute(wk_adjoint<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->L.wp.smem_adj)
            : cudaFuncSetAttribute(wk_adjoint<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->L.wp.smem_adj);
        if (e1 != cudaSuccess || e2 != cudaSuccess) return fail(h, -4, "shared-memory opt-in of the wavefront kernels failed");
        // row tables per tile row: entry r+1 <-> padded row r = -1 .. py, guard values of the virtual pole rows
        std::vector<double> wt((size_t)h->L.p2 * h->L.wp.wtab_stride, 0.0);
        const double* T6 = h->h_tab.data();
        for (int b = 0; b < h->L.p2; ++b) {
            const Sub& sb = h->L.hs[(size_t)b * h->L.p1];
            for (int q = 0; q < sb.py + 2; ++q) {
                const int gj = sb.ej0 - sb.gys + q - 1;
                const int cj = gj < 0 ? 0 : (gj >= nlat ? nlat - 1 : gj);
                double* t = &wt[(size_t)b * h->L.wp.wtab_stride + (size_t)q * 8];
                t[0] = T6[cj]; t[1] = T6[nlat + cj]; t[2] = T6[2 * nlat + cj]; t[3] = T6[3 * nlat + cj];
                t[4] = gj < 0 ? 1.0 : T6[4 * nlat + cj];
                t[5] = gj >= nlat ? 1.0 : T6[5 * nlat + cj];
                t[6] = h->mp.dtcm * t[4]; t[7] = h->mp.dtcm * t[5];
            }
        }
        CU(cudaMemcpyAsync(h->L.wp.wtab, wt.data(), sizeof(double) * wt.size(), cudaMemcpyHostToDevice, h->stream));
        CU(cudaStreamSynchronize(h->stream));
    }
    rc = upload_chunk_masks(h, h->L);
    if (rc) return rc;
    if (h->L.fp.enabled) {
        h->h_ctab.assign(6 * (size_t)FK_CTAB, 0.0);
        if (fused_upload_tables(h->stream, h->h_tab.data(), nlat, h->h_ctab.data(), h->d_ctab))
            return fail(h, -4, "upload of the row tables failed");
    }
    fused_teardown(h->stream, h->L.fp);         // (a second set_workspace on the same handle)
    rc = fused_setup(h->stream, h->L.fp, h->L.dsubs);
    if (rc) return fail(h, -4, "fused kernel setup failed (persisting-L2 window)");
    h->have_ws = true; h->have_bg = false; h->G.have_obs = h->L.have_obs = false;
    return sync_check(h);
}

int dd4dvar_set_background(dd4dvar_t h, const double* d_xb, const double h_sigma_b[3])
{
    if (!h || !d_xb || !h_sigma_b) return fail(h, -1, "set_background: null argument");
    if (!h->have_ws) return fail(h, -3, "set_background before set_workspace");
    for (int f = 0; f < 3; ++f) {
        if (!(h_sigma_b[f] > 0)) return fail(h, -1, "set_background: sigma_b must be positive");
        h->cp.sb[f] = h_sigma_b[f]; h->cp.ib[f] = 1.0 / (h_sigma_b[f] * h_sigma_b[f]);
    }
    Layout& G = h->G; Layout& L = h->L;
    const size_t n3 = 3 * (size_t)h->grid.nlon * h->grid.nlat;
    CU(cudaMemcpyAsync(G.xbs, d_xb, sizeof(double) * n3, cudaMemcpyDeviceToDevice, h->stream));
    CU(cudaMemcpyAsync(G.x, d_xb, sizeof(double) * n3, cudaMemcpyDeviceToDevice, h->stream));
    // Alg 1 l.452: u^b = M(u_0^b)
    forward_generic(h, G, nullptr);
    // l.455: u_ji^0 = u_ji^b; local stores = restricted background trajectory
    for (int lev = 0; lev <= h->win.nsteps; ++lev)
        LAUNCH(xk_restrict_level, cell_grid(L), NT_GK, L.dsubs, h->grid.nlon, h->grid.nlat, lev,
               G.traj + (size_t)lev * n3, L.traj, L.xbs, L.x);
    CU(cudaMemsetAsync(L.w, 0, sizeof(double) * L.ctot, h->stream));
    exchange(h, L);
    h->have_bg = true;
    return sync_check(h);
}

size_t dd4dvar_obs_workspace_bytes(dd4dvar_t h, long long n_obs_total)
{
    if (!h || n_obs_total < 0) return 0;
    const size_t per = 4 + 4 + 8 + 8 + 8 + 8;
    size_t nb = (size_t)n_obs_total * (1 + 2 * (size_t)h->L.maxcov);
    return nb * per + (size_t)(h->G.otot + h->L.otot + 8) * 8 + 4096;
}

static int bin_observations(dd4dvar_t h, Layout& L, int n_times, const int* levels, const long long* offs,
                            const int* idx, const double* val, Arena& ar, bool weights)
{
    const int nlon = h->grid.nlon, nlat = h->grid.nlat;
    const long long n1 = (long long)nlon * nlat;
    std::vector<long long> start(L.otot + 1, 0);
    // Def 8 l.239: restriction of H^(k) to Delta_j x Omega_i = the observations inside it
    auto visit = [&](auto&& fn) {
        for (int t = 0; t < n_times; ++t) {
            const int lev = levels[t];
            for (long long qq = offs[t]; qq < offs[t + 1]; ++qq) {
                const int f = (int)(idx[qq] / n1); const long long c = idx[qq] % n1;
                const int gj = (int)(c / nlon), gi = (int)(c % nlon);
                int ntime = 0;
                for (int jw = 0; jw < L.q; ++jw) if (lev >= L.wb[jw] && lev <= L.wb[jw + 1]) ++ntime;
                for (int jw = 0; jw < L.q; ++jw) {
                    if (lev < L.wb[jw] || lev > L.wb[jw + 1]) continue;
                    for (int cb = 0; cb < L.nrowcov[gj]; ++cb)
                        for (int ca = 0; ca < L.ncolcov[gi]; ++ca) {
                            const int k = (jw * L.p2 + L.rowcov[4 * gj + cb]) * L.p1 + L.colcov[4 * gi + ca];
                            const Sub& s = L.hs[k];
                            const int li = imod(gi - s.ei0, nlon), lj = gj - s.ej0;
                            const double wt = weights ? 1.0 / (double)(L.ncolcov[gi] * L.nrowcov[gj]) / (double)ntime : 1.0;
                            fn(s.ooff + (lev - s.s), f * s.ncell + lj * s.ex + li, val[qq], wt, f);
                        }
                }
            }
        }
    };
    visit([&](long long bin, int, double, double, int) { ++start[bin + 1]; });
    for (long long b = 0; b < L.otot; ++b) start[b + 1] += start[b];
    const long long nb = start[L.otot];
    std::vector<long long> fill(start.begin(), start.end() - 1);
    std::vector<int> oi(nb + 1), ol(nb + 1); std::vector<double> oy(nb + 1), oc(nb + 1);
    visit([&](long long bin, int lidx, double y, double wt, int f) {
        const long long p = fill[bin]++;
        oi[p] = lidx; oy[p] = y; oc[p] = h->cp.lambda * wt / (h->sig_o[f] * h->sig_o[f]);
    });
    // inside a bin: ascending (tile row, field, column), the order in which the wavefront kernels
    // meet the cells; obs_lj = packed (tile row, field, column) of every entry
    {
        std::vector<long long> sub_of_bin(L.otot, 0);
        for (int k = 0; k < L.nsub; ++k)
            for (int n = 0; n <= L.hs[k].W + 1; ++n) if (L.hs[k].ooff + n < L.otot) sub_of_bin[L.hs[k].ooff + n] = k;
        std::vector<long long> ord; std::vector<int> ti; std::vector<double> ty, tc;
        for (long long b = 0; b < L.otot; ++b) {
            const long long a0 = start[b], a1 = start[b + 1];
            if (a1 <= a0) continue;
            const Sub& sb = L.hs[sub_of_bin[b]];
            auto key = [&](long long p) {
                const int f = oi[p] / sb.ncell, c = oi[p] - f * sb.ncell;
                const int lj = c / sb.ex, li = c - lj * sb.ex;
                return ((long long)lj * 3 + f) * sb.ex + li;
            };
            ord.resize(a1 - a0);
            for (long long p = a0; p < a1; ++p) ord[p - a0] = p;
            std::sort(ord.begin(), ord.end(), [&](long long p, long long q) { return key(p) < key(q); });
            ti.resize(a1 - a0); ty.resize(a1 - a0); tc.resize(a1 - a0);
            for (long long p = 0; p < a1 - a0; ++p) { ti[p] = oi[ord[p]]; ty[p] = oy[ord[p]]; tc[p] = oc[ord[p]]; }
            for (long long p = 0; p < a1 - a0; ++p) {
                oi[a0 + p] = ti[p]; oy[a0 + p] = ty[p]; oc[a0 + p] = tc[p];
                {   // packed (tile row << 12) | (field << 8) | column  (wave kernels: no divisions)
                    const int f = ti[p] / sb.ncell, c = ti[p] - f * sb.ncell;
                    const int lj = c / sb.ex, li = c - lj * sb.ex;
                    ol[a0 + p] = (lj << 12) | (f << 8) | li;
                }
            }
        }
    }
    L.obs_start = ar.take<long long>(L.otot + 1);
    L.obs_idx = ar.take<int>(nb + 1); L.obs_lj = ar.take<int>(nb + 1);
    L.obs_y = ar.take<double>(nb + 1); L.obs_c = ar.take<double>(nb + 1); L.obs_r = ar.take<double>(nb + 1);
    L.obs_rt = ar.take<double>(nb + 1);
    if (ar.off > ar.cap) return fail(h, -1, "set_observations: observation workspace too small");
    CU(cudaMemcpyAsync(L.obs_lj, ol.data(), sizeof(int) * (nb + 1), cudaMemcpyHostToDevice, h->stream));
    CU(cudaMemsetAsync(L.obs_r, 0, sizeof(double) * (nb + 1), h->stream));
    CU(cudaMemsetAsync(L.obs_rt, 0, sizeof(double) * (nb + 1), h->stream));
    CU(cudaMemcpyAsync(L.obs_start, start.data(), sizeof(long long) * (L.otot + 1), cudaMemcpyHostToDevice, h->stream));
    CU(cudaMemcpyAsync(L.obs_idx, oi.data(), sizeof(int) * (nb + 1), cudaMemcpyHostToDevice, h->stream));
    CU(cudaMemcpyAsync(L.obs_y, oy.data(), sizeof(double) * (nb + 1), cudaMemcpyHostToDevice, h->stream));
    CU(cudaMemcpyAsync(L.obs_c, oc.data(), sizeof(double) * (nb + 1), cudaMemcpyHostToDevice, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    L.have_obs = true;
    return 0;
}

int dd4dvar_set_observations(dd4dvar_t h, int n_times, const int* h_levels, const long long* h_offsets,
                             const int* d_index, const double* d_value, const double h_sigma_o[3],
                             void* d_obs_ws, size_t obs_ws_bytes)
{
    if (!h || n_times < 0 || !h_sigma_o) return fail(h, -1, "set_observations: bad argument");
    if (!h->have_ws) return fail(h, -3, "set_observations before set_workspace");
    if (n_times > 0 && (!h_levels || !h_offsets || !d_index || !d_value || !d_obs_ws))
        return fail(h, -1, "set_observations: null argument");
    for (int f = 0; f < 3; ++f) {
        if (!(h_sigma_o[f] > 0)) return fail(h, -1, "set_observations: sigma_o must be positive");
        h->sig_o[f] = h_sigma_o[f];
    }
    const long long tot = n_times ? h_offsets[n_times] : 0;
    if (n_times && obs_ws_bytes < dd4dvar_obs_workspace_bytes(h, tot))
        return fail(h, -1, "set_observations: observation workspace too small");
    std::vector<int> idx(tot + 1); std::vector<double> val(tot + 1);
    if (tot) {
        CU(cudaMemcpyAsync(idx.data(), d_index, sizeof(int) * tot, cudaMemcpyDeviceToHost, h->stream));
        CU(cudaMemcpyAsync(val.data(), d_value, sizeof(double) * tot, cudaMemcpyDeviceToHost, h->stream));
        CU(cudaStreamSynchronize(h->stream));
    }
    const long long n3 = 3LL * h->grid.nlon * h->grid.nlat;
    for (int t = 0; t < n_times; ++t) {
        if (h_levels[t] < 0 || h_levels[t] > h->win.nsteps || (t && h_levels[t] <= h_levels[t - 1]))
            return fail(h, -1, "set_observations: levels must be strictly ascending inside [0, nsteps]");
        if (h_offsets[t + 1] < h_offsets[t]) return fail(h, -1, "set_observations: offsets must ascend");
        for (long long q = h_offsets[t]; q < h_offsets[t + 1]; ++q) {
            if (idx[q] < 0 || idx[q] >= n3) return fail(h, -1, "set_observations: index out of range");
            if (q > h_offsets[t] && idx[q] <= idx[q - 1])
                return fail(h, -1, "set_observations: indices must be strictly ascending inside a level");
        }
    }
    Arena ar; ar.base = (char*)d_obs_ws; ar.cap = obs_ws_bytes;
    int rc = 0;
    if (n_times == 0) { h->G.have_obs = h->L.have_obs = false; return 0; }
    rc = bin_observations(h, h->G, n_times, h_levels, h_offsets, idx.data(), val.data(), ar, false);
    if (!rc) rc = bin_observations(h, h->L, n_times, h_levels, h_offsets, idx.data(), val.data(), ar, true);
    return rc;
}

int dd4dvar_eval_global(dd4dvar_t h, const double* d_x0, double* h_cost, double* d_grad)
{
    if (!h || !d_x0 || !h_cost) return fail(h, -1, "eval_global: null argument");
    if (!h->have_bg) return fail(h, -3, "eval_global before set_background");
    Layout& G = h->G;
    const size_t n3 = 3 * (size_t)h->grid.nlon * h->grid.nlat;
    CU(cudaMemcpyAsync(G.x, d_x0, sizeof(double) * n3, cudaMemcpyDeviceToDevice, h->stream));
    sweep(h, G, d_grad != nullptr, nullptr, G.Jev, nullptr);
    CU(cudaMemcpyAsync(h_cost, G.Jev, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    if (d_grad) CU(cudaMemcpyAsync(d_grad, G.gx, sizeof(double) * n3, cudaMemcpyDeviceToDevice, h->stream));
    int rc = sync_check(h);
    if (rc) return rc;
    if (!isfinite(*h_cost)) return fail(h, -5, "eval_global: non-finite cost");
    return 0;
}

int dd4dvar_eval_local(dd4dvar_t h, const double* d_controls, double* h_costs, double* h_parts, double* d_grads)
{
    if (!h || !d_controls || !h_costs) return fail(h, -1, "eval_local: null argument");
    if (!h->have_bg) return fail(h, -3, "eval_local before set_background");
    Layout& L = h->L;
    CU(cudaMemcpyAsync(L.x, d_controls, sizeof(double) * L.ctot, cudaMemcpyDeviceToDevice, h->stream));
    sweep(h, L, d_grads != nullptr, nullptr, L.Jev, nullptr);
    CU(cudaMemcpyAsync(h_costs, L.Jev, sizeof(double) * L.nsub, cudaMemcpyDeviceToHost, h->stream));
    if (h_parts) CU(cudaMemcpyAsync(h_parts, L.parts, sizeof(double) * 5 * L.nsub, cudaMemcpyDeviceToHost, h->stream));
    if (d_grads) CU(cudaMemcpyAsync(d_grads, L.gx, sizeof(double) * L.ctot, cudaMemcpyDeviceToDevice, h->stream));
    int rc = sync_check(h);
    if (rc) return rc;
    for (int k = 0; k < L.nsub; ++k)
        if (!isfinite(h_costs[k])) return fail(h, -5, "eval_local: non-finite cost");
    return 0;
}

int dd4dvar_eval_local_host(dd4dvar_t h, const double* h_controls, double* h_costs, double* h_grads)
{
    if (!h || !h_controls || !h_costs) return fail(h, -1, "eval_local_host: null argument");
    if (!h->have_bg) return fail(h, -3, "eval_local_host before set_background");
    Layout& L = h->L;
    if (L.nsub < 64) {                          // small problems: one copy in, one sweep, one copy out
        CU(cudaMemcpyAsync(L.x, h_controls, sizeof(double) * L.ctot, cudaMemcpyHostToDevice, h->stream));
        sweep(h, L, h_grads != nullptr, nullptr, L.Jev, nullptr);
        CU(cudaMemcpyAsync(h_costs, L.Jev, sizeof(double) * L.nsub, cudaMemcpyDeviceToHost, h->stream));
        if (h_grads) CU(cudaMemcpyAsync(h_grads, L.gx, sizeof(double) * L.ctot, cudaMemcpyDeviceToHost, h->stream));
    } else {
        // Subdomains are independent inside one evaluation (all neighbour data is frozen), so the evaluation runs in
        // EH_CHUNKS chunks of consecutive subdomains: the host -> device copy of chunk c+1 and the device -> host copy
        // of chunk c-1 overlap the sweep of chunk c (two copy streams, masked sweeps on the caller's stream).
        if (!h->s_h2d) {
            CU(cudaStreamCreateWithFlags(&h->s_h2d, cudaStreamNonBlocking));
            CU(cudaStreamCreateWithFlags(&h->s_d2h, cudaStreamNonBlocking));
            CU(cudaEventCreateWithFlags(&h->ev_in, cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&h->ev_out, cudaEventDisableTiming));
            for (int c = 0; c < EH_CHUNKS; ++c) {
                CU(cudaEventCreateWithFlags(&h->ev_h2d[c], cudaEventDisableTiming));
                CU(cudaEventCreateWithFlags(&h->ev_sw[c], cudaEventDisableTiming));
            }
        }
        CU(cudaEventRecord(h->ev_in, h->stream));                       // the copies start after the caller's earlier work
        CU(cudaStreamWaitEvent(h->s_h2d, h->ev_in, 0));
        CU(cudaStreamWaitEvent(h->s_d2h, h->ev_in, 0));
        int kb[EH_CHUNKS + 1];
        eh_bounds(L, kb);
        auto off = [&](int k) { return k < L.nsub ? L.hs[k].coff : L.ctot; };
        for (int c = 0; c < EH_CHUNKS; ++c) {
            const long long o0 = off(kb[c]), o1 = off(kb[c + 1]);
            CU(cudaMemcpyAsync(L.x + o0, h_controls + o0, sizeof(double) * (o1 - o0), cudaMemcpyHostToDevice, h->s_h2d));
            CU(cudaEventRecord(h->ev_h2d[c], h->s_h2d));
        }
        for (int c = 0; c < EH_CHUNKS; ++c) {
            const long long o0 = off(kb[c]), o1 = off(kb[c + 1]);
            CU(cudaStreamWaitEvent(h->stream, h->ev_h2d[c], 0));
            sweep(h, L, h_grads != nullptr, L.cmask + (size_t)c * L.nsub, L.Jev, nullptr);
            CU(cudaEventRecord(h->ev_sw[c], h->stream));
            CU(cudaStreamWaitEvent(h->s_d2h, h->ev_sw[c], 0));
            CU(cudaMemcpyAsync(h_costs + kb[c], L.Jev + kb[c], sizeof(double) * (kb[c + 1] - kb[c]), cudaMemcpyDeviceToHost, h->s_d2h));
            if (h_grads) CU(cudaMemcpyAsync(h_grads + o0, L.gx + o0, sizeof(double) * (o1 - o0), cudaMemcpyDeviceToHost, h->s_d2h));
        }
        CU(cudaEventRecord(h->ev_out, h->s_d2h));
        CU(cudaStreamWaitEvent(h->stream, h->ev_out, 0));
    }
    int rc = sync_check(h);
    if (rc) return rc;
    for (int k = 0; k < L.nsub; ++k)
        if (!isfinite(h_costs[k])) return fail(h, -5, "eval_local_host: non-finite cost");
    return 0;
}

int dd4dvar_sweep_async(dd4dvar_t h, int mode)
{
    if (!h || mode < 0 || mode > 2) return -1;
    if (!h->have_bg) return fail(h, -3, "sweep_async before set_background");
    if (mode == 2) adjoint_only(h, h->L, nullptr, nullptr);
    else sweep(h, h->L, mode == 1, nullptr, h->L.Jev, nullptr);
    return 0;
}

int dd4dvar_get_controls(dd4dvar_t h, double* d_controls)
{
    if (!h || !d_controls) return fail(h, -1, "get_controls: null argument");
    if (!h->have_bg) return fail(h, -3, "get_controls before set_background");
    CU(cudaMemcpyAsync(d_controls, h->L.xfrozen, sizeof(double) * h->L.ctot, cudaMemcpyDeviceToDevice, h->stream));
    return sync_check(h);
}

int dd4dvar_get_trajectory(dd4dvar_t h, int level, double* d_out)
{
    if (!h || !d_out || level < 0 || level > h->win.nsteps) return fail(h, -1, "get_trajectory: bad argument");
    if (!h->have_bg) return fail(h, -3, "get_trajectory before set_background");
    const int n1 = h->grid.nlon * h->grid.nlat;
    LAUNCH(xk_gather, (n1 + 255) / 256, 256, h->L.dsubs, h->L.geo, 0, level, h->L.traj, d_out);
    return sync_check(h);
}

int dd4dvar_get_local_trajectory(dd4dvar_t h, int sub, double* d_out)
{
    if (!h || !d_out || sub < 0 || sub >= h->L.nsub) return fail(h, -1, "get_local_trajectory: bad argument");
    if (!h->have_bg) return fail(h, -3, "get_local_trajectory before set_background");
    const Sub& s = h->L.hs[sub];
    CU(cudaMemcpyAsync(d_out, h->L.traj + s.toff, sizeof(double) * (size_t)(s.W + 1) * 3 * s.ncell,
                       cudaMemcpyDeviceToDevice, h->stream));
    return sync_check(h);
}

int dd4dvar_forecast(dd4dvar_t h, const double* d_x0, int n_levels, const int* h_levels, double* d_out)
{
    if (!h || !d_x0 || n_levels < 0 || (n_levels && (!h_levels || !d_out))) return fail(h, -1, "forecast: bad argument");
    if (!h->have_ws) return fail(h, -3, "forecast before set_workspace");
    Layout& G = h->G;
    const size_t n3 = 3 * (size_t)h->grid.nlon * h->grid.nlat;
    for (int q = 0; q < n_levels; ++q)
        if (h_levels[q] < 0 || h_levels[q] > h->win.nsteps || (q && h_levels[q] < h_levels[q - 1]))
            return fail(h, -1, "forecast: levels must ascend inside [0, nsteps]");
    CU(cudaMemcpyAsync(G.x, d_x0, sizeof(double) * n3, cudaMemcpyDeviceToDevice, h->stream));
    forward_generic(h, G, nullptr);
    for (int q = 0; q < n_levels; ++q)
        CU(cudaMemcpyAsync(d_out + (size_t)q * n3, G.traj + (size_t)h_levels[q] * n3, sizeof(double) * n3,
                           cudaMemcpyDeviceToDevice, h->stream));
    return sync_check(h);
}

// Algorithm 1 l.443-472 (additive outer iteration R16, fixed iteration count R17)
int dd4dvar_run(dd4dvar_t h, int outer_iters, double* d_analysis, double* h_history)
{
    if (!h || outer_iters < 0 || !d_analysis || !h_history) return fail(h, -1, "run: bad argument");
    if (!h->have_bg) return fail(h, -3, "run before set_background");
    Layout& L = h->L; Layout& G = h->G;
    const int n1 = h->grid.nlon * h->grid.nlat;
    const int nsub = L.nsub;
    const int* own = L.sharded ? L.own : nullptr;       // sharded runs: only the subdomains of the owned windows move
    LbfgsP lp; lp.m = h->opt.lbfgs_m; lp.max_bt = h->opt.max_backtrack; lp.c1 = h->opt.armijo_c1; lp.ctot = L.ctot;
    h->h_tmp.resize(std::max(nsub, 8));
    int rc;
    auto sumJ = [&](const double* dJ, double* out) -> int {
        CU(cudaMemcpyAsync(h->h_tmp.data(), dJ, sizeof(double) * nsub, cudaMemcpyDeviceToHost, h->stream));
        int r = sync_check(h); if (r) return r;
        long double sacc = 0; for (int k = 0; k < nsub; ++k) sacc += h->h_tmp[k];
        *out = (double)sacc; return 0;
    };
    auto gather_and_cost = [&](double* out) -> int {
        if (!h->history_global) { *out = nan(""); return 0; }
        LAUNCH(xk_gather, (n1 + 255) / 256, 256, L.dsubs, L.geo, 1, 0, L.xfrozen, G.x);
        return global_cost(h, out);
    };
    h->ph_kind.clear();
    for (double& v : h->ph_ms) v = 0.0;
    ph_mark(h, PH_JGLOBAL);
    if ((rc = gather_and_cost(&h_history[0]))) return rc;
    ph_mark(h, PH_LBFGS);
    CU(cudaMemsetAsync(L.st.nactive, 0, 2 * sizeof(int), h->stream));
    h_history[1] = 0.0; h_history[2] = 0.0;
    const dim3 vgrid(std::min(64, (3 * L.maxncell + 255) / 256), nsub);
    if (outer_iters == 0) {
        LAUNCH(lk_trial, vgrid, 256, L.dsubs, own, h->cp, (const double*)nullptr, L.w,
               (const double*)nullptr, L.xbs, (double*)nullptr, L.x);
        ph_mark(h, PH_SWEEP);
        sweep(h, L, false, own, L.st.J, nullptr);
        ph_mark(h, PH_LBFGS);
        if ((rc = sumJ(L.st.J, &h_history[1]))) return rc;
    }
    for (int l = 1; l <= outer_iters; ++l) {
        // local functional changed: clear the history (R10), evaluate J_ji and its gradient at w
        CU(cudaMemsetAsync(L.st.nh, 0, sizeof(int) * nsub, h->stream));
        CU(cudaMemsetAsync(L.st.head, 0, sizeof(int) * nsub, h->stream));
        if (own) CU(cudaMemcpyAsync(L.st.done, L.notown, sizeof(int) * nsub, cudaMemcpyDeviceToDevice, h->stream));
        else CU(cudaMemsetAsync(L.st.done, 0, sizeof(int) * nsub, h->stream));
        LAUNCH(lk_trial, vgrid, 256, L.dsubs, own, h->cp, (const double*)nullptr, L.w,
               (const double*)nullptr, L.xbs, (double*)nullptr, L.x);
        ph_mark(h, PH_SWEEP);
        sweep(h, L, true, own, L.st.J, L.g);
        ph_mark(h, PH_LBFGS);
        if (l == 1 && (rc = sumJ(L.st.J, &h_history[1]))) return rc;
        for (int it = 0; it < h->opt.n_inner; ++it) {
            LAUNCH(lk_direction<NT_LB>, nsub * LK_CL, NT_LB, L.dsubs, lp, L.st, L.g, L.S, L.Y, L.d);
            for (int b = 0; b <= lp.max_bt; ++b) {
                CU(cudaMemsetAsync(L.st.nactive, 0, sizeof(int), h->stream));
                LAUNCH(lk_trial, vgrid, 256, L.dsubs, L.st.active, h->cp, L.st.t, L.w, L.d, L.xbs, L.wt, L.x);
                ph_mark(h, PH_SWEEP);
                sweep(h, L, false, L.st.active, L.st.Jt, nullptr);
                ph_mark(h, PH_LBFGS);
                LAUNCH(lk_lscheck, (nsub + 127) / 128, 128, nsub, lp, L.st);
                int nact[2] = { 0, 0 };
                CU(cudaMemcpyAsync(nact, L.st.nactive, 2 * sizeof(int), cudaMemcpyDeviceToHost, h->stream));
                if ((rc = sync_check(h))) return rc;
                if (nact[1]) return fail(h, -5, "run: non-finite gradient");
                if (nact[0] == 0) break;
            }
            // gradient at the accepted points (their trajectories are still in the store)
            ph_mark(h, PH_SWEEP);
            adjoint_only(h, L, L.st.ok, L.gn);
            ph_mark(h, PH_LBFGS);
            LAUNCH(lk_update<NT_LB>, nsub * LK_CL, NT_LB, L.dsubs, lp, L.st, L.w, L.wt, L.g, L.gn, L.S, L.Y);
        }
        // one more forward sweep so that the stored trajectory belongs to the accepted iterate
        LAUNCH(lk_trial, vgrid, 256, L.dsubs, own, h->cp, (const double*)nullptr, L.w,
               (const double*)nullptr, L.xbs, (double*)nullptr, L.x);
        ph_mark(h, PH_SWEEP);
        sweep(h, L, false, own, L.Jev, nullptr);
        ph_mark(h, PH_LBFGS);
        if ((rc = sumJ(L.st.J, &h_history[3 * l + 1]))) return rc;
        ph_mark(h, PH_EXCH);
        exchange(h, L);
        CU(cudaMemcpyAsync(h->h_tmp.data(), L.dmax, sizeof(double) * nsub, cudaMemcpyDeviceToHost, h->stream));
        if ((rc = sync_check(h))) return rc;
        double dl = 0; for (int k = 0; k < nsub; ++k) dl = std::max(dl, h->h_tmp[k]);
        h_history[3 * l + 2] = dl;
        ph_mark(h, PH_JGLOBAL);
        if ((rc = gather_and_cost(&h_history[3 * l]))) return rc;
        ph_mark(h, PH_LBFGS);
        if ((h->history_global && !isfinite(h_history[3 * l])) || !isfinite(h_history[3 * l + 1])) return fail(h, -5, "run: non-finite cost");
    }
    ph_mark(h, PH_OTHER);
    LAUNCH(xk_gather, (n1 + 255) / 256, 256, L.dsubs, L.geo, 1, 0, L.xfrozen, d_analysis);
    ph_mark(h, -1);
    rc = sync_check(h);
    ph_collect(h);
    return rc;
}

int dd4dvar_set_phase_timing(dd4dvar_t h, int on)
{
    if (!h) return -1;
    h->ph_on = on != 0;
    return 0;
}

int dd4dvar_get_phase_ms(dd4dvar_t h, double h_out[5])
{
    if (!h || !h_out) return -1;
    for (int q = 0; q < 5; ++q) h_out[q] = h->ph_ms[q];
    return 0;
}

// ---- Gauss-Newton local minimiser (gn_kernels.cuh): wavefront layouts only ------------------
namespace {
// Hp (w-space) = H_GN pw about the trajectory the last forward sweep stored
int gn_apply(dd4dvar_t h, Layout& L, const double* pw, double* Hp)
{
    const dim3 pgrid((L.maxnpad + 255) / 256, L.nsub);
    LAUNCH(tk_init, pgrid, 256, L.dsubs, h->cp, pw, L.Zp, L.Za);
    double* din = L.Zp; double* dout = L.Za;
    const size_t smem = sizeof(double) * TK_SMEM_DOUBLES;
    const bool generic = L.path != 5;
    if (generic) LAUNCH(tk_store, cell_grid(L), NT_GK, L.dsubs, 0, din, L.gn_dtraj);
    for (int n = 0; n < L.Wmax; ++n) {
        tk_step<<<dim3(L.ntiles, L.nsub), SK_NT, smem, h->stream>>>(L.dsubs, n, h->mp, L.traj, L.ghost, din, dout, L.tiles_x);
        ++h->launches;
        if (generic) LAUNCH(tk_store, cell_grid(L), NT_GK, L.dsubs, n + 1, dout, L.gn_dtraj);
        else if (L.have_obs)
            LAUNCH(tk_obs, dim3(2, L.nsub), 128, L.dsubs, n + 1, L.obs_start, L.obs_lj, L.obs_c, dout, L.obs_rt);
        std::swap(din, dout);
    }
    if (generic) {
        // generic layouts: the adjoint sweep of the per-stage / block-tiled kernels with the tangent-linear trajectory as
        // the source of every forcing term (obs_rt serves as the all-zero observation vector: it is never written here)
        LAUNCH(gn_scale_x, dim3(std::min(32, (3 * L.maxncell + 255) / 256), L.nsub), 256, L.dsubs, h->cp, pw, L.gn_gx);
        adjoint_generic(h, L, nullptr, Hp, L.gn_dtraj, L.gn_gx, L.gn_zero, L.obs_rt, nullptr);
        return 0;
    }
    LAUNCH(ck_gn, L.nsub, 256, L.dsubs, L.dnb, L.geo, h->cp, pw, L.Zp, L.Za, L.have_obs ? L.obs_start : nullptr,
           L.obs_lj, L.obs_c, L.obs_rt, L.gn_gx, L.gn_lamW);
    WkArgs a = wave_args(h, L, nullptr, nullptr, nullptr);
    a.obs_r = L.obs_rt; a.lamW = L.gn_lamW; a.gx = L.gn_gx;
    if (L.wp.K == 2) wk_adjoint<2><<<L.wp.grid, WK_NT, L.wp.smem_adj, h->stream>>>(a);
    else wk_adjoint<3><<<L.wp.grid, WK_NT, L.wp.smem_adj, h->stream>>>(a);
    ++h->launches;
    LAUNCH(ck_scale_grad, dim3(std::min(32, (3 * L.maxncell + 255) / 256), L.nsub), 256, L.dsubs, (const int*)nullptr,
           h->cp, L.gn_gx, Hp);
    return 0;
}
}  // namespace

int dd4dvar_gn_hessvec(dd4dvar_t h, const double* d_controls, const double* d_p, double* d_out)
{
    if (!h || !d_controls || !d_p || !d_out) return fail(h, -1, "gn_hessvec: null argument");
    if (!h->have_bg) return fail(h, -3, "gn_hessvec before set_background");
    Layout& L = h->L;
    if (L.path == 2 || L.path == 4 || !L.gn_Hp) return fail(h, -2, "gn_hessvec: the Gauss-Newton solver is served by the wavefront (path 5) and the generic kernels (path 1, 3)");
    if (h->overlap_levels) return fail(h, -2, "gn_hessvec: not available with dd4dvar_set_overlap_levels (the all-level overlap penalty has no Gauss-Newton path)");
    CU(cudaMemcpyAsync(L.x, d_controls, sizeof(double) * L.ctot, cudaMemcpyDeviceToDevice, h->stream));
    sweep(h, L, false, nullptr, L.Jev, nullptr);
    int rc = gn_apply(h, L, d_p, L.gn_Hp);
    if (rc) return rc;
    CU(cudaMemcpyAsync(d_out, L.gn_Hp, sizeof(double) * L.ctot, cudaMemcpyDeviceToDevice, h->stream));
    return sync_check(h);
}

// Algorithm 1 l.443-472 with the local minimiser of Algorithms 5-7 (Gauss-Newton + CG in w-space)
int dd4dvar_run_gn(dd4dvar_t h, int outer_iters, int n_gn, int n_cg, double* d_analysis, double* h_history)
{
    if (!h || outer_iters < 0 || n_gn < 0 || n_cg < 0 || !d_analysis || !h_history) return fail(h, -1, "run_gn: bad argument");
    if (!h->have_bg) return fail(h, -3, "run_gn before set_background");
    Layout& L = h->L; Layout& G = h->G;
    if (L.path == 2 || L.path == 4 || !L.gn_Hp) return fail(h, -2, "run_gn: the Gauss-Newton solver is served by the wavefront (path 5) and the generic kernels (path 1, 3)");
    if (L.sharded) return fail(h, -2, "run_gn: not available in sharded runs (dd4dvar_set_owned_windows)");
    if (h->overlap_levels) return fail(h, -2, "run_gn: not available with dd4dvar_set_overlap_levels (the all-level overlap penalty has no Gauss-Newton path)");
    const int n1 = h->grid.nlon * h->grid.nlat;
    const int nsub = L.nsub;
    h->h_tmp.resize(std::max(nsub, 8));
    int rc;
    auto sumJ = [&](const double* dJ, double* out) -> int {
        CU(cudaMemcpyAsync(h->h_tmp.data(), dJ, sizeof(double) * nsub, cudaMemcpyDeviceToHost, h->stream));
        int r = sync_check(h); if (r) return r;
        long double sacc = 0; for (int k = 0; k < nsub; ++k) sacc += h->h_tmp[k];
        *out = (double)sacc; return 0;
    };
    auto gather_and_cost = [&](double* out) -> int {
        if (!h->history_global) { *out = nan(""); return 0; }
        LAUNCH(xk_gather, (n1 + 255) / 256, 256, L.dsubs, L.geo, 1, 0, L.xfrozen, G.x);
        return global_cost(h, out);
    };
    const dim3 vgrid(std::min(64, (3 * L.maxncell + 255) / 256), nsub);
    auto controls_from_w = [&]() {
        LAUNCH(lk_trial, vgrid, 256, L.dsubs, (const int*)nullptr, h->cp, (const double*)nullptr, L.w,
               (const double*)nullptr, L.xbs, (double*)nullptr, L.x);
    };
    if ((rc = gather_and_cost(&h_history[0]))) return rc;
    h_history[1] = 0.0; h_history[2] = 0.0;
    if (outer_iters == 0) {
        controls_from_w();
        sweep(h, L, false, nullptr, L.st.J, nullptr);
        if ((rc = sumJ(L.st.J, &h_history[1]))) return rc;
    }
    double* dw = L.d; double* rv = L.wt; double* pv = L.gn;
    for (int l = 1; l <= outer_iters; ++l) {
        for (int it = 0; it < n_gn; ++it) {
            controls_from_w();
            sweep(h, L, true, nullptr, L.st.J, L.g);                   // J_ji, g = sigma_b grad_x J_ji, trajectory
            if (l == 1 && it == 0 && (rc = sumJ(L.st.J, &h_history[1]))) return rc;
            LAUNCH(gn_cg_init, nsub, GN_NT, L.dsubs, L.g, dw, rv, pv, L.st.t, L.st.trial);
            for (int c = 0; c < n_cg; ++c) {
                if ((rc = gn_apply(h, L, pv, L.gn_Hp))) return rc;
                LAUNCH(gn_cg_update, nsub, GN_NT, L.dsubs, L.gn_Hp, dw, rv, pv, L.st.t, L.st.trial);
            }
            LAUNCH(gn_add, vgrid, 256, L.dsubs, L.w, dw);
        }
        // forward sweep at the final iterate: its trajectory is what the neighbours see next
        controls_from_w();
        sweep(h, L, false, nullptr, L.st.J, nullptr);
        if (l == 1 && n_gn == 0 && (rc = sumJ(L.st.J, &h_history[1]))) return rc;
        if ((rc = sumJ(L.st.J, &h_history[3 * l + 1]))) return rc;
        exchange(h, L);
        CU(cudaMemcpyAsync(h->h_tmp.data(), L.dmax, sizeof(double) * nsub, cudaMemcpyDeviceToHost, h->stream));
        if ((rc = sync_check(h))) return rc;
        double dl = 0; for (int k = 0; k < nsub; ++k) dl = std::max(dl, h->h_tmp[k]);
        h_history[3 * l + 2] = dl;
        if ((rc = gather_and_cost(&h_history[3 * l]))) return rc;
        if ((h->history_global && !isfinite(h_history[3 * l])) || !isfinite(h_history[3 * l + 1])) return fail(h, -5, "run_gn: non-finite cost");
    }
    LAUNCH(xk_gather, (n1 + 255) / 256, 256, L.dsubs, L.geo, 1, 0, L.xfrozen, d_analysis);
    return sync_check(h);
}

int dd4dvar_set_bg_weight(dd4dvar_t h, double w_later)
{
    if (!h || !(w_later >= 0.0)) return fail(h, -1, "set_bg_weight: weight must be >= 0");
    h->cp.bgw = w_later;
    return 0;
}

// ---- sharded runs: one process per GPU owns a block of time windows -------------
int dd4dvar_set_owned_windows(dd4dvar_t h, int j0, int j1)
{
    if (!h) return -1;
    if (!h->have_ws) return fail(h, -3, "set_owned_windows before set_workspace");
    Layout& L = h->L;
    if (j0 < 0 || j1 > L.q || j0 >= j1) return fail(h, -1, "set_owned_windows: need 0 <= j0 < j1 <= q_time");
    std::vector<int> own(L.nsub), notown(L.nsub);
    for (int k = 0; k < L.nsub; ++k) { own[k] = L.hs[k].jw >= j0 && L.hs[k].jw < j1; notown[k] = !own[k]; }
    CU(cudaMemcpyAsync(L.own, own.data(), sizeof(int) * L.nsub, cudaMemcpyHostToDevice, h->stream));
    CU(cudaMemcpyAsync(L.notown, notown.data(), sizeof(int) * L.nsub, cudaMemcpyHostToDevice, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    L.sharded = !(j0 == 0 && j1 == L.q); L.own_j0 = j0; L.own_j1 = j1;
    return 0;
}

int dd4dvar_exchange_buffer(dd4dvar_t h, int which, void** d_ptr, long long* count)
{
    if (!h || !d_ptr || !count) return -1;
    if (!h->have_ws) return fail(h, -3, "exchange_buffer before set_workspace");
    Layout& L = h->L;
    switch (which) {
    case 0: *d_ptr = L.xfrozen; *count = L.ctot; return 0;
    case 1: *d_ptr = L.pred_end; *count = L.ctot; return 0;
    default: return fail(h, -1, "exchange_buffer: which = 0 (frozen controls) or 1 (predecessor end states)");
    }
}

int dd4dvar_get_local_stats(dd4dvar_t h, double* h_J, double* h_dmax)
{
    if (!h || !h_J || !h_dmax) return fail(h, -1, "get_local_stats: null argument");
    if (!h->have_bg) return fail(h, -3, "get_local_stats before set_background");
    CU(cudaMemcpyAsync(h_J, h->L.st.J, sizeof(double) * h->L.nsub, cudaMemcpyDeviceToHost, h->stream));
    CU(cudaMemcpyAsync(h_dmax, h->L.dmax, sizeof(double) * h->L.nsub, cudaMemcpyDeviceToHost, h->stream));
    return sync_check(h);
}

int dd4dvar_gather_analysis(dd4dvar_t h, double* d_analysis)
{
    if (!h || !d_analysis) return fail(h, -1, "gather_analysis: null argument");
    if (!h->have_bg) return fail(h, -3, "gather_analysis before set_background");
    const int n1 = h->grid.nlon * h->grid.nlat;
    LAUNCH(xk_gather, (n1 + 255) / 256, 256, h->L.dsubs, h->L.geo, 1, 0, h->L.xfrozen, d_analysis);
    return sync_check(h);
}

int dd4dvar_set_overlap_levels(dd4dvar_t h, int on)
{
    if (!h) return -1;
    if (h->have_bg) return fail(h, -3, "set_overlap_levels after set_background");
    if (on && h->L.path != 1 && h->L.path != 3)
        return fail(h, -2, "set_overlap_levels: served by the generic kernels only (create with opts.path = 1)");
    h->overlap_levels = on != 0;
    return 0;
}

int dd4dvar_set_history_global(dd4dvar_t h, int on)
{
    if (!h) return -1;
    h->history_global = on != 0;
    return 0;
}

int dd4dvar_measure_peaks(void* cuda_stream, double h_out[6])
{
    if (!h_out) return -1;
    return measure_peaks((cudaStream_t)cuda_stream, h_out);
}

int dd4dvar_num_subdomains(dd4dvar_t h) { return h ? h->L.nsub : -1; }

int dd4dvar_subdomain_info(dd4dvar_t h, int sub, int out[16])
{
    if (!h || !out || sub < 0 || sub >= h->L.nsub) return fail(h, -1, "subdomain_info: bad argument");
    const Sub& s = h->L.hs[sub];
    const int v[16] = { s.a, s.b, s.jw, s.oi0, s.oi1, s.oj0, s.oj1, s.ei0, s.ej0, s.ex, s.ey, s.gx, s.gys, s.gyn, s.s, s.s + s.W };
    memcpy(out, v, sizeof(v));
    return 0;
}

long long dd4dvar_control_offset(dd4dvar_t h, int sub)
{
    if (!h || sub < 0 || sub > h->L.nsub) return -1;
    return sub == h->L.nsub ? h->L.ctot : h->L.hs[sub].coff;
}

int dd4dvar_active_path(dd4dvar_t h) { return h ? h->L.path : -1; }
long long dd4dvar_launch_count(dd4dvar_t h) { return h ? h->launches : -1; }
const char* dd4dvar_last_error(dd4dvar_t h) { return h ? h->err.c_str() : "null handle"; }
void dd4dvar_destroy(dd4dvar_t h)
{
    if (!h) return;
    fused_teardown(h->stream, h->L.fp);
    for (cudaEvent_t e : h->ph_ev) cudaEventDestroy(e);
    if (h->s_h2d) {
        cudaStreamSynchronize(h->s_h2d); cudaStreamSynchronize(h->s_d2h);
        cudaStreamDestroy(h->s_h2d); cudaStreamDestroy(h->s_d2h);
        cudaEventDestroy(h->ev_in); cudaEventDestroy(h->ev_out);
        for (int c = 0; c < EH_CHUNKS; ++c) { cudaEventDestroy(h->ev_h2d[c]); cudaEventDestroy(h->ev_sw[c]); }
    }
    delete h;
}

}  // extern "C"

// ================================================== forecast without device allocation ====
// dd4dvar_forecast_static (include/dd4dvar.h): the model forecast of dd4dvar_forecast for callers that have no way
// of obtaining device memory for the library: no handle, no workspace.  Everything the step kernel needs beyond the
// caller's input and output -- the six row tables of the model and the time levels it steps between -- lives in ONE
// array that is part of the library image.  The array is reserved on every GPU that loads libdd4dvar.so, for the life
// of the process, whether or not this entry point is ever called; hence its modest, fixed size.
#include <mutex>

#define DD_STATIC_DOUBLES ((size_t)DD4DVAR_STATIC_SCRATCH_BYTES / sizeof(double))
static __device__ __align__(256) double dd_static_scratch[DD_STATIC_DOUBLES];

namespace {

// `dd_static_scratch` in HOST code is only a handle for the runtime's symbol look-up, not an address a kernel could
// use.  The device address differs per GPU; it is asked for once per device (with that device current) and kept here.
constexpr int DD_STATIC_MAXDEV = 64;
double* g_static_base[DD_STATIC_MAXDEV] = {};
std::mutex g_static_mutex;

int static_scratch_base(double** out, std::string& err)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { err = std::string("cudaGetDevice: ") + cudaGetErrorString(e); return -4; }
    if (dev < 0 || dev >= DD_STATIC_MAXDEV) { err = "device ordinal beyond the table of dd4dvar_forecast_static"; return -4; }
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_base[dev]) {
        double* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, dd_static_scratch);
        if (e != cudaSuccess || !p) {
            err = std::string("cudaGetSymbolAddress(dd_static_scratch): ") + cudaGetErrorString(e);
            return -4;
        }
        g_static_base[dev] = p;
    }
    *out = g_static_base[dev];
    return 0;
}

// The same row tables as dd4dvar_create builds (O1: eq (60)-(62) l.945-954, cell-centred rows R2, clamped metric R3,
// dt folded in), written out a second time so that the handle-based path stays untouched.  tab: [6][nlat].
void static_row_tables(const dd4dvar_grid& g, double dt, std::vector<double>& tab, ModelP& mp)
{
    const int nlat = g.nlat;
    const double PI = 3.14159265358979323846;
    const double dlam = 2.0 * PI / g.nlon, dth = PI / nlat, a = g.radius;
    std::vector<double> mc(nlat);
    tab.assign(6 * (size_t)nlat, 0.0);
    double* dtcz = &tab[0]; double* gdtcz = &tab[nlat]; double* dtf = &tab[2 * (size_t)nlat];
    double* dtt = &tab[3 * (size_t)nlat]; double* rp = &tab[4 * (size_t)nlat]; double* rm = &tab[5 * (size_t)nlat];
    for (int j = 0; j < nlat; ++j) {
        const double th = -0.5 * PI + (j + 0.5) * dth, c = cos(th);
        mc[j] = c > g.cos_clamp ? c : g.cos_clamp;
        const double cz = 1.0 / (2.0 * a * dlam * mc[j]);
        dtcz[j] = dt * cz; gdtcz[j] = g.gravity * dt * cz;
        dtf[j] = dt * 2.0 * g.omega * sin(th);
        dtt[j] = dt * sin(th) / (a * mc[j]);
    }
    for (int j = 0; j < nlat; ++j) {
        rp[j] = (j + 1 < nlat ? mc[j + 1] : mc[j]) / mc[j];
        rm[j] = (j > 0 ? mc[j - 1] : mc[j]) / mc[j];
    }
    const double cm = 1.0 / (2.0 * a * dth);
    mp.nlon = g.nlon; mp.nlat = nlat; mp.kap = g.diffusion;
    mp.dtcm = dt * cm; mp.gdtcm = g.gravity * dt * cm;
}

// Variant of sk_forward_step (step_kernels.cuh) for the undecomposed grid: the descriptor of the one region travels as a
// kernel argument, the row tables behind `m` and the time levels behind `levels` are inside dd_static_scratch.  The step
// reads level `slot` and writes level `slot + 1` of `levels` ([.][3][nlat][nlon]); the region has no ghost ring
// (periodic in longitude, pole walls), so no ghost store is read.  Same tile code as the handle-based forecast.
__global__ void __launch_bounds__(SK_NT) sk_forward_step_static(Sub s, int slot, ModelP m, double* levels, int tiles_x)
{
    __shared__ double smf[SK_FWD_SMEM_DOUBLES];
    sk_forward_tile(s, blockIdx.x % tiles_x, blockIdx.x / tiles_x, slot, m, levels, levels, smf,
                    smf + 3 * (SK_TY + 6) * (SK_TX + 6), smf + 3 * (SK_TY + 6) * (SK_TX + 6) + 3 * (SK_TY + 4) * (SK_TX + 4));
}

int static_fail(char* h_err, size_t err_len, int code, const std::string& msg)
{
    if (h_err && err_len) { strncpy(h_err, msg.c_str(), err_len - 1); h_err[err_len - 1] = 0; }
    return code;
}

}  // namespace

extern "C" int dd4dvar_forecast_static(const dd4dvar_grid* grid, const dd4dvar_window* window, const double* d_x0,
                                       int n_levels, const int* h_levels, double* d_out, void* cuda_stream,
                                       char* h_err, size_t err_len)
{
    if (h_err && err_len) h_err[0] = 0;
    if (!grid || !window || !d_x0 || n_levels < 0 || (n_levels && (!h_levels || !d_out)))
        return static_fail(h_err, err_len, -1, "forecast_static: null argument");
    if (grid->nlon < 3 || grid->nlat < 2 || window->nsteps < 1 || !(grid->radius > 0))
        return static_fail(h_err, err_len, -1, "forecast_static: bad grid or window");
    for (int q = 0; q < n_levels; ++q)
        if (h_levels[q] < 0 || h_levels[q] > window->nsteps || (q && h_levels[q] < h_levels[q - 1]))
            return static_fail(h_err, err_len, -1, "forecast_static: levels must ascend inside [0, nsteps]");
    // size check first: tables (rounded up to 256 bytes) + at least two time levels must fit the static array
    const size_t n3 = 3 * (size_t)grid->nlon * grid->nlat;
    const size_t tab_doubles = (6 * (size_t)grid->nlat + 31) & ~size_t(31);
    const size_t cap = tab_doubles < DD_STATIC_DOUBLES ? (DD_STATIC_DOUBLES - tab_doubles) / n3 : 0;
    if (cap < 2) {
        char msg[256];
        snprintf(msg, sizeof msg,
                 "forecast_static: a %d x %d grid needs %zu bytes of scratch (row tables + two time levels), the static "
                 "array holds %zu; use dd4dvar_forecast with a caller-allocated workspace",
                 grid->nlon, grid->nlat, sizeof(double) * (tab_doubles + 2 * n3), (size_t)DD4DVAR_STATIC_SCRATCH_BYTES);
        return static_fail(h_err, err_len, -6, msg);
    }
    Layout G;
    if (build_layout(G, grid->nlon, grid->nlat, window->nsteps, 1, 1, 1, 0))
        return static_fail(h_err, err_len, -2, "forecast_static: the grid cannot be laid out");
    std::string err;
    double* base = nullptr;
    int rc = static_scratch_base(&base, err);      // first call on a device: symbol look-up (set-up; keep it out of stream capture)
    if (rc) return static_fail(h_err, err_len, rc, "forecast_static: " + err);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaError_t e;
#define CUS(call)                                                                                              \
    do {                                                                                                       \
        e = (call);                                                                                            \
        if (e != cudaSuccess)                                                                                  \
            return static_fail(h_err, err_len, -4, std::string("forecast_static: " #call ": ") + cudaGetErrorString(e)); \
    } while (0)
    // Nothing in the array has to start at zero: the tables and level 0 are rewritten here, and every later level is
    // written in full by the step that produces it before anything reads it.  What the last call left is overwritten.
    std::vector<double> tab;
    ModelP mp{};
    static_row_tables(*grid, window->dt, tab, mp);
    const int nlat = grid->nlat;
    mp.dtcz = base; mp.gdtcz = base + nlat; mp.dtf = base + 2 * (size_t)nlat;
    mp.dtt = base + 3 * (size_t)nlat; mp.rp = base + 4 * (size_t)nlat; mp.rm = base + 5 * (size_t)nlat;
    double* levels = base + tab_doubles;
    CUS(cudaMemcpyAsync(base, tab.data(), sizeof(double) * tab.size(), cudaMemcpyHostToDevice, st));
    CUS(cudaMemcpyAsync(levels, d_x0, sizeof(double) * n3, cudaMemcpyDeviceToDevice, st));
    const Sub s = G.hs[0];
    int q = 0;
    while (q < n_levels && h_levels[q] == 0) {
        CUS(cudaMemcpyAsync(d_out + (size_t)q * n3, levels, sizeof(double) * n3, cudaMemcpyDeviceToDevice, st));
        ++q;
    }
    // the array holds `cap` consecutive levels; when the next step would run past its end, the newest level moves to
    // slot 0 and the stepping goes on from there
    size_t slot = 0;
    for (int n = 0; n < window->nsteps && q < n_levels; ++n) {
        if (slot + 1 == cap) {
            CUS(cudaMemcpyAsync(levels, levels + slot * n3, sizeof(double) * n3, cudaMemcpyDeviceToDevice, st));
            slot = 0;
        }
        sk_forward_step_static<<<G.ntiles, SK_NT, 0, st>>>(s, (int)slot, mp, levels, G.tiles_x);
        CUS(cudaGetLastError());
        ++slot;
        while (q < n_levels && h_levels[q] == n + 1) {
            CUS(cudaMemcpyAsync(d_out + (size_t)q * n3, levels + slot * n3, sizeof(double) * n3, cudaMemcpyDeviceToDevice, st));
            ++q;
        }
    }
    CUS(cudaStreamSynchronize(st));
    CUS(cudaGetLastError());
#undef CUS
    return 0;
}
