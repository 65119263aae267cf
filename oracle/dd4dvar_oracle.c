/*
 * dd4dvar_oracle.c -- CPU ORACLE for the space-time decomposed 4D-Var (DD-4DVar) hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no
 * code, header, table or constant generator with the CUDA path (paper_2205_06649_b200/csrc).
 *
 * Plain, slow, fp64, written step by step from /root/reference/PAPER.md (arXiv 2205.06649) and
 * the readings listed in DESIGN.md (R1..R20, mirroring SURVEY.md §8(c) Q1..Q20).  No blocking,
 * fusion or reordering beyond what the cited passage states; sums use long double accumulators.
 * Compile with -ffp-contract=off (no FMA contraction).  OpenMP only over independent subdomains
 * (and over rows of one stage of the global step); results do not depend on the thread count.
 *
 * What it computes (citations are PAPER.md line numbers):
 *   O1  grid and row tables                      eq (60)-(62) l.945-954, eq (67) l.976-980
 *   O2  one model step Phi (split scheme)        l.971-989 member p=q=1, alpha=0; R3
 *   O3  tangent-linear and adjoint of Phi        Def 1 l.86-87; eq (3) l.91; eq (4) l.98
 *   O4  global functional J and gradient         Def 2 eq (5)-(6) l.105-114
 *   O5  space-time decomposition                 Def 3 l.128-154; Def 16 l.755-763; eq (70) l.1024
 *   O6  restriction weights                      Def 4 l.164-170
 *   O7  regularised local functional J_ji        Def 11 eq (16)-(17) l.251-267; Def 13 eq (23)-(25)
 *                                                l.326-344; overlap operator eq (20)-(22) l.294-322
 *   O8  local minimiser (L-BFGS)                 Remark 3 l.595; l.941; eq (44) l.630-634
 *   O9  outer loop, exchange, gather             Algorithm 1 l.443-472; eq (12)-(13) l.194-201
 *
 * PINS (tests/test_oracle_*.py, -m "not gpu"): rest-state fixed point, closed-form linear
 * dispersion of zonal/meridional gravity waves and inertial oscillation, one-step FTCS
 * advection-diffusion amplification, O(Delta^2) drift of the balanced zonal flow, TLM Taylor
 * remainder, adjoint dot-product identity eq (3), finite-difference gradients, the per-point
 * closed-form minimiser when Phi = identity, sum of weights = 1 (eq 12), sum_ji J_ji(u^b) =
 * J(u^b) (eq 19), 1x1x1 layout = plain global 4D-Var, L-BFGS vs a dense solve, local sweep with
 * exact ghost data = global trajectory, the consensus fixed point of the outer loop when
 * Phi = identity.  "parity unpinned": the final DD analysis values on the SWE configs (the
 * paper prints none; PAPER.md:995 defers validation to its ref [12]).
 */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#define NF 3          /* fields h,u,v */
#define GHOST 3       /* stencil reach of one full step: stage A 1 + h1 1 + u1/v1 1 (R14) */

typedef struct {
    int nlon, nlat;
    double a, Omega, g, cos_clamp, kappa, dt;
    double cm;                 /* 1/(2 a dtheta) */
    double *f, *t, *cz, *rp, *rm, *mc;
} Model;

/* ------------------------------------------------------------------ O1: row tables ------- */
static void model_tables(Model* m)
{
    const double PI = 3.14159265358979323846;
    int n = m->nlat;
    double dlam = 2.0 * PI / m->nlon, dth = PI / n;
    m->f = malloc(sizeof(double) * n); m->t = malloc(sizeof(double) * n);
    m->cz = malloc(sizeof(double) * n); m->rp = malloc(sizeof(double) * n);
    m->rm = malloc(sizeof(double) * n); m->mc = malloc(sizeof(double) * n);
    for (int j = 0; j < n; ++j) {
        double th = -0.5 * PI + (j + 0.5) * dth;          /* cell-centred rows (R2) */
        double c = cos(th);
        m->mc[j] = c > m->cos_clamp ? c : m->cos_clamp;   /* clamped metric (R3) */
        m->f[j] = 2.0 * m->Omega * sin(th);
        m->t[j] = sin(th) / (m->a * m->mc[j]);
        m->cz[j] = 1.0 / (2.0 * m->a * dlam * m->mc[j]);
    }
    for (int j = 0; j < n; ++j) {
        double mn = j + 1 < n ? m->mc[j + 1] : m->mc[j];  /* beyond a pole row: that row's m */
        double ms = j > 0 ? m->mc[j - 1] : m->mc[j];
        m->rp[j] = mn / m->mc[j];
        m->rm[j] = ms / m->mc[j];
    }
    m->cm = 1.0 / (2.0 * m->a * dth);
}
static void model_free(Model* m)
{ free(m->f); free(m->t); free(m->cz); free(m->rp); free(m->rm); free(m->mc); }

/* ------------------------------------------------------------------ O2: the step ---------
 * A "region" is a rectangular array [3][py][px] whose row 0 is global row joff.  A side is
 * either closed by the model's own rule (periodic in longitude; reflective pole wall: ghost row
 * = edge row with v negated, re-applied at every sub-stage, R4) or open: then the valid range
 * shrinks by one cell per sub-stage (stage A: 1, h1: 2, u1/v1: 3 = GHOST).
 * Global grid: per_x = wall_s = wall_n = 1.  Local padded tile: open sides carry the ghost ring.
 */
typedef struct { int px, py, joff, per_x, wall_s, wall_n; } Region;

static void stage_range(const Region* r, int k, int* i0, int* i1, int* j0, int* j1)
{
    int ox = r->per_x ? 0 : k;
    *i0 = ox; *i1 = r->px - ox;
    *j0 = r->wall_s ? 0 : k;
    *j1 = r->wall_n ? r->py : r->py - k;
}
/* neighbour indices of (i,j); sN/sS = mirror sign that applies to v when the neighbour is a
 * reflected pole ghost row (h and u use +1 there). */
static inline void nbrs(const Region* r, int i, int j, int* iE, int* iW, int* jN, int* jS,
                        double* sN, double* sS)
{
    *iE = i + 1; *iW = i - 1;
    if (r->per_x) { if (*iE == r->px) *iE = 0; if (*iW < 0) *iW = r->px - 1; }
    *jN = j + 1; *jS = j - 1; *sN = 1.0; *sS = 1.0;
    if (r->wall_n && j == r->py - 1) { *jN = j; *sN = -1.0; }
    if (r->wall_s && j == 0)         { *jS = j; *sS = -1.0; }
}
#define AT(p, fld, j, i) ((p)[((size_t)(fld) * r->py + (j)) * r->px + (i)])

/* Z0 -> Za (stage A, valid on range 1) -> Z1 (h1 valid on range 2, u1 and v1 on range 3). */
static void region_forward(const Model* m, const Region* r, const double* Z0, double* Za,
                           double* Z1)
{
    const double dt = m->dt, kap = m->kappa, cm = m->cm, g = m->g;
    int i0, i1, j0, j1;
    /* Stage A: advection of h,u,v by (u0,v0), forward Euler, plus index-space diffusion */
    stage_range(r, 1, &i0, &i1, &j0, &j1);
#pragma omp parallel for if (r->py > 256)
    for (int j = j0; j < j1; ++j) {
        double cz = m->cz[r->joff + j];
        for (int i = i0; i < i1; ++i) {
            int iE, iW, jN, jS; double sN, sS;
            nbrs(r, i, j, &iE, &iW, &jN, &jS, &sN, &sS);
            double u0 = AT(Z0, 1, j, i), v0 = AT(Z0, 2, j, i);
            for (int fl = 0; fl < NF; ++fl) {
                double mN = fl == 2 ? sN : 1.0, mS = fl == 2 ? sS : 1.0;
                double x = AT(Z0, fl, j, i);
                double xE = AT(Z0, fl, j, iE), xW = AT(Z0, fl, j, iW);
                double xN = mN * AT(Z0, fl, jN, i), xS = mS * AT(Z0, fl, jS, i);
                AT(Za, fl, j, i) = x - dt * (cz * u0 * (xE - xW) + cm * v0 * (xN - xS))
                                 + kap * (xE + xW + xN + xS - 4.0 * x);
            }
        }
    }
    /* Stage B, height first */
    stage_range(r, 2, &i0, &i1, &j0, &j1);
#pragma omp parallel for if (r->py > 256)
    for (int j = j0; j < j1; ++j) {
        int gj = r->joff + j;
        double cz = m->cz[gj], rp = m->rp[gj], rm = m->rm[gj];
        for (int i = i0; i < i1; ++i) {
            int iE, iW, jN, jS; double sN, sS;
            nbrs(r, i, j, &iE, &iW, &jN, &jS, &sN, &sS);
            double ha = AT(Za, 0, j, i);
            double vaN = sN * AT(Za, 2, jN, i), vaS = sS * AT(Za, 2, jS, i);
            AT(Z1, 0, j, i) = ha - dt * ha * (cz * (AT(Za, 1, j, iE) - AT(Za, 1, j, iW))
                                              + cm * (rp * vaN - rm * vaS));
        }
    }
    /* then u, then v (forward-backward) */
    stage_range(r, 3, &i0, &i1, &j0, &j1);
#pragma omp parallel for if (r->py > 256)
    for (int j = j0; j < j1; ++j) {
        int gj = r->joff + j;
        double cz = m->cz[gj], f = m->f[gj], t = m->t[gj];
        for (int i = i0; i < i1; ++i) {
            int iE, iW, jN, jS; double sN, sS;
            nbrs(r, i, j, &iE, &iW, &jN, &jS, &sN, &sS);
            double ua = AT(Za, 1, j, i), va = AT(Za, 2, j, i);
            double u1 = ua + dt * (-g * cz * (AT(Z1, 0, j, iE) - AT(Z1, 0, j, iW))
                                   + (f + t * ua) * va);
            double v1 = va + dt * (-g * cm * (AT(Z1, 0, jN, i) - AT(Z1, 0, jS, i))
                                   - (f + t * u1) * u1);
            AT(Z1, 1, j, i) = u1;
            AT(Z1, 2, j, i) = v1;
        }
    }
}

/* ------------------------------------------------------------------ O3: TLM --------------
 * dZ0 given on the whole region (zero where the state is frozen), dZ1 as Z1's ranges. */
static void region_tlm(const Model* m, const Region* r, const double* Z0, const double* Za,
                       const double* Z1, const double* dZ0, double* dZa, double* dZ1)
{
    const double dt = m->dt, kap = m->kappa, cm = m->cm, g = m->g;
    int i0, i1, j0, j1;
    stage_range(r, 1, &i0, &i1, &j0, &j1);
    for (int j = j0; j < j1; ++j) {
        double cz = m->cz[r->joff + j];
        for (int i = i0; i < i1; ++i) {
            int iE, iW, jN, jS; double sN, sS;
            nbrs(r, i, j, &iE, &iW, &jN, &jS, &sN, &sS);
            double u0 = AT(Z0, 1, j, i), v0 = AT(Z0, 2, j, i);
            double du0 = AT(dZ0, 1, j, i), dv0 = AT(dZ0, 2, j, i);
            for (int fl = 0; fl < NF; ++fl) {
                double mN = fl == 2 ? sN : 1.0, mS = fl == 2 ? sS : 1.0;
                double xE = AT(Z0, fl, j, iE), xW = AT(Z0, fl, j, iW);
                double xN = mN * AT(Z0, fl, jN, i), xS = mS * AT(Z0, fl, jS, i);
                double dx = AT(dZ0, fl, j, i);
                double dxE = AT(dZ0, fl, j, iE), dxW = AT(dZ0, fl, j, iW);
                double dxN = mN * AT(dZ0, fl, jN, i), dxS = mS * AT(dZ0, fl, jS, i);
                AT(dZa, fl, j, i) = dx
                    - dt * (cz * du0 * (xE - xW) + cz * u0 * (dxE - dxW)
                            + cm * dv0 * (xN - xS) + cm * v0 * (dxN - dxS))
                    + kap * (dxE + dxW + dxN + dxS - 4.0 * dx);
            }
        }
    }
    stage_range(r, 2, &i0, &i1, &j0, &j1);
    for (int j = j0; j < j1; ++j) {
        int gj = r->joff + j;
        double cz = m->cz[gj], rp = m->rp[gj], rm = m->rm[gj];
        for (int i = i0; i < i1; ++i) {
            int iE, iW, jN, jS; double sN, sS;
            nbrs(r, i, j, &iE, &iW, &jN, &jS, &sN, &sS);
            double ha = AT(Za, 0, j, i), dha = AT(dZa, 0, j, i);
            double D = cz * (AT(Za, 1, j, iE) - AT(Za, 1, j, iW))
                     + cm * (rp * sN * AT(Za, 2, jN, i) - rm * sS * AT(Za, 2, jS, i));
            double dD = cz * (AT(dZa, 1, j, iE) - AT(dZa, 1, j, iW))
                      + cm * (rp * sN * AT(dZa, 2, jN, i) - rm * sS * AT(dZa, 2, jS, i));
            AT(dZ1, 0, j, i) = dha - dt * (dha * D + ha * dD);
        }
    }
    stage_range(r, 3, &i0, &i1, &j0, &j1);
    for (int j = j0; j < j1; ++j) {
        int gj = r->joff + j;
        double cz = m->cz[gj], f = m->f[gj], t = m->t[gj];
        for (int i = i0; i < i1; ++i) {
            int iE, iW, jN, jS; double sN, sS;
            nbrs(r, i, j, &iE, &iW, &jN, &jS, &sN, &sS);
            double ua = AT(Za, 1, j, i), va = AT(Za, 2, j, i), u1 = AT(Z1, 1, j, i);
            double dua = AT(dZa, 1, j, i), dva = AT(dZa, 2, j, i);
            double du1 = dua + dt * (-g * cz * (AT(dZ1, 0, j, iE) - AT(dZ1, 0, j, iW))
                                     + t * dua * va + (f + t * ua) * dva);
            double dv1 = dva + dt * (-g * cm * (AT(dZ1, 0, jN, i) - AT(dZ1, 0, jS, i))
                                     - (f + 2.0 * t * u1) * du1);
            AT(dZ1, 1, j, i) = du1;
            AT(dZ1, 2, j, i) = dv1;
        }
    }
}

/* ------------------------------------------------------------------ O3: adjoint ----------
 * Transposes of the TLM statements, in reverse order (eq (4) l.98), scatter form.
 * L1 = adjoint of (h1,u1,v1), non-zero only on range 3; out L0 on the whole region.
 * Work: A (adjoint of Za) and HB (adjoint of h1), both [py][px]-sized, zeroed here. */
static void region_adjoint(const Model* m, const Region* r, const double* Z0, const double* Za,
                           const double* Z1, const double* L1, double* A, double* HB, double* UB,
                           double* L0)
{
    const double dt = m->dt, kap = m->kappa, cm = m->cm, g = m->g;
    size_t n1 = (size_t)r->px * r->py;
    int i0, i1, j0, j1;
    memset(A, 0, sizeof(double) * NF * n1);
    memset(HB, 0, sizeof(double) * n1);
    memset(UB, 0, sizeof(double) * n1);
    memset(L0, 0, sizeof(double) * NF * n1);
#define A_(fl, j, i) A[((size_t)(fl) * r->py + (j)) * r->px + (i)]
#define HB_(j, i) HB[(size_t)(j) * r->px + (i)]
#define UB_(j, i) UB[(size_t)(j) * r->px + (i)]
    stage_range(r, 3, &i0, &i1, &j0, &j1);
    for (int j = j0; j < j1; ++j)
        for (int i = i0; i < i1; ++i) { HB_(j, i) = AT(L1, 0, j, i); UB_(j, i) = AT(L1, 1, j, i); }
    /* v1 = va + dt*( -g cm (h1N - h1S) - (f + t u1) u1 ) */
    for (int j = j0; j < j1; ++j) {
        int gj = r->joff + j;
        double f = m->f[gj], t = m->t[gj];
        for (int i = i0; i < i1; ++i) {
            int iE, iW, jN, jS; double sN, sS;
            nbrs(r, i, j, &iE, &iW, &jN, &jS, &sN, &sS);
            double vb = AT(L1, 2, j, i), u1 = AT(Z1, 1, j, i);
            A_(2, j, i) += vb;
            HB_(jN, i) += -dt * g * cm * vb;          /* h mirrors with +1 */
            HB_(jS, i) += dt * g * cm * vb;
            UB_(j, i) += -dt * (f + 2.0 * t * u1) * vb;
        }
    }
    /* u1 = ua + dt*( -g cz (h1E - h1W) + (f + t ua) va ) */
    for (int j = j0; j < j1; ++j) {
        int gj = r->joff + j;
        double cz = m->cz[gj], f = m->f[gj], t = m->t[gj];
        for (int i = i0; i < i1; ++i) {
            int iE, iW, jN, jS; double sN, sS;
            nbrs(r, i, j, &iE, &iW, &jN, &jS, &sN, &sS);
            double ub = UB_(j, i), ua = AT(Za, 1, j, i), va = AT(Za, 2, j, i);
            A_(1, j, i) += ub * (1.0 + dt * t * va);
            A_(2, j, i) += ub * dt * (f + t * ua);
            HB_(j, iE) += -dt * g * cz * ub;
            HB_(j, iW) += dt * g * cz * ub;
        }
    }
    /* h1 = ha - dt*ha*D,  D = cz (uaE - uaW) + cm (rp vaN - rm vaS) */
    stage_range(r, 2, &i0, &i1, &j0, &j1);
    for (int j = j0; j < j1; ++j) {
        int gj = r->joff + j;
        double cz = m->cz[gj], rp = m->rp[gj], rm = m->rm[gj];
        for (int i = i0; i < i1; ++i) {
            int iE, iW, jN, jS; double sN, sS;
            nbrs(r, i, j, &iE, &iW, &jN, &jS, &sN, &sS);
            double hb = HB_(j, i), ha = AT(Za, 0, j, i);
            double D = cz * (AT(Za, 1, j, iE) - AT(Za, 1, j, iW))
                     + cm * (rp * sN * AT(Za, 2, jN, i) - rm * sS * AT(Za, 2, jS, i));
            double c = -dt * ha * hb;
            A_(0, j, i) += hb * (1.0 - dt * D);
            A_(1, j, iE) += c * cz;
            A_(1, j, iW) -= c * cz;
            A_(2, jN, i) += sN * c * cm * rp;
            A_(2, jS, i) -= sS * c * cm * rm;
        }
    }
    /* stage A */
    stage_range(r, 1, &i0, &i1, &j0, &j1);
    for (int j = j0; j < j1; ++j) {
        double cz = m->cz[r->joff + j];
        for (int i = i0; i < i1; ++i) {
            int iE, iW, jN, jS; double sN, sS;
            nbrs(r, i, j, &iE, &iW, &jN, &jS, &sN, &sS);
            double u0 = AT(Z0, 1, j, i), v0 = AT(Z0, 2, j, i);
            for (int fl = 0; fl < NF; ++fl) {
                double mN = fl == 2 ? sN : 1.0, mS = fl == 2 ? sS : 1.0;
                double xb = A_(fl, j, i);
                double xE = AT(Z0, fl, j, iE), xW = AT(Z0, fl, j, iW);
                double xN = mN * AT(Z0, fl, jN, i), xS = mS * AT(Z0, fl, jS, i);
                AT(L0, fl, j, i) += xb * (1.0 - 4.0 * kap);
                AT(L0, fl, j, iE) += xb * (-dt * cz * u0 + kap);
                AT(L0, fl, j, iW) += xb * (dt * cz * u0 + kap);
                AT(L0, fl, jN, i) += mN * xb * (-dt * cm * v0 + kap);
                AT(L0, fl, jS, i) += mS * xb * (dt * cm * v0 + kap);
                AT(L0, 1, j, i) += -dt * cz * (xE - xW) * xb;
                AT(L0, 2, j, i) += -dt * cm * (xN - xS) * xb;
            }
        }
    }
#undef A_
#undef HB_
#undef UB_
}
#undef AT

/* ------------------------------------------------------------------ handle ---------------- */
typedef struct {
    int a, b, jw;                 /* tile column, tile row, window */
    int oi0, oi1, oj0, oj1;       /* owned ranges (global cells) */
    int ei0, ej0, ex, ey;         /* extended tile: origin (column unwrapped, may be <0), size */
    int gx, gys, gyn;             /* ghost widths (0 = closed side) */
    int s, e;                     /* window levels s..e inclusive */
    long ncell;
} Sub;

typedef struct { int tidx, fld; long cell; double y; } LocObs;   /* one local observation */

typedef struct {
    Model m;
    int nsteps;
    int p1, p2, q, o;
    double mu, lambda;
    int ovl_levels;   /* (25c) case 1 on every level of the window (eq (21) l.300 read literally: O_ik maps onto Delta_j x
                       * (Omega_i n Omega_k)), not on the control level only (reading R12, the default 0) */
    double bgw;   /* weight of (25a) in windows j > 0 (0 = only at t_0, reading R7, the default; 1 = in every window as (25a) is printed) */
    int lbfgs_m, n_inner, max_bt; double c1;
    int nsub; Sub* sub;
    int *colown, *rowown;         /* owner tile column / row of a global column / row */
    int *ncolcov, *colcov;        /* tiles whose extended range covers a global column (<=4) */
    int *nrowcov, *rowcov;
    int* wb;                      /* window boundaries s_0..s_Q */
    /* background */
    int have_bg; double sig_b[3]; double* xb; double* ubtraj;   /* [(N+1)][3][nlat][nlon] */
    /* observations (global) */
    int have_obs; int ntimes; int* olev; long long* ooff; int* oidx; double* oval; double sig_o[3];
    long* nlocobs; LocObs** locobs;      /* binned per subdomain */
    /* frozen (previous outer iteration) and current local data; NULL = "the background" */
    double **w_prev, **x_prev, **traj_prev;
    double **w_cur, **x_cur, **traj_cur;
    char err[256];
} DD;

static int imod(int a, int n) { int r = a % n; return r < 0 ? r + n : r; }

/* O5: owned ranges floor(a*n/p) .. floor((a+1)*n/p) (ragged allowed, R9); extended = owned +- o,
 * periodic in longitude, truncated at the pole walls; p1 = 1: the tile wraps onto itself. */
static int build_decomposition(DD* d)
{
    int nlon = d->m.nlon, nlat = d->m.nlat, N = d->nsteps, o = d->o;
    if (d->p1 < 1 || d->p2 < 1 || d->q < 1 || o < 0 || d->q > N) return -2;
    d->wb = malloc(sizeof(int) * (d->q + 1));
    for (int j = 0; j <= d->q; ++j) d->wb[j] = (int)(((long)j * N) / d->q);
    d->nsub = d->p1 * d->p2 * d->q;
    d->sub = calloc(d->nsub, sizeof(Sub));
    d->colown = malloc(sizeof(int) * nlon); d->rowown = malloc(sizeof(int) * nlat);
    d->ncolcov = calloc(nlon, sizeof(int)); d->colcov = malloc(sizeof(int) * 4 * nlon);
    d->nrowcov = calloc(nlat, sizeof(int)); d->rowcov = malloc(sizeof(int) * 4 * nlat);
    for (int jw = 0; jw < d->q; ++jw)
        for (int b = 0; b < d->p2; ++b)
            for (int a = 0; a < d->p1; ++a) {
                Sub* s = &d->sub[(jw * d->p2 + b) * d->p1 + a];
                s->a = a; s->b = b; s->jw = jw;
                s->oi0 = (int)(((long)a * nlon) / d->p1); s->oi1 = (int)(((long)(a + 1) * nlon) / d->p1);
                s->oj0 = (int)(((long)b * nlat) / d->p2); s->oj1 = (int)(((long)(b + 1) * nlat) / d->p2);
                if (s->oi1 <= s->oi0 || s->oj1 <= s->oj0) return -2;
                if (d->p1 == 1) { s->ei0 = 0; s->ex = nlon; s->gx = 0; }
                else { s->ei0 = s->oi0 - o; s->ex = s->oi1 - s->oi0 + 2 * o; s->gx = GHOST; }
                if (s->ex > nlon) return -2;
                int j0 = s->oj0 - o, j1 = s->oj1 + o;
                if (j0 < 0) j0 = 0;
                if (j1 > nlat) j1 = nlat;
                s->ej0 = j0; s->ey = j1 - j0;
                s->gys = j0 == 0 ? 0 : GHOST;
                s->gyn = j1 == nlat ? 0 : GHOST;
                if (j0 - s->gys < 0 || j1 + s->gyn > nlat) return -2;   /* ghost ring off the grid */
                s->s = d->wb[jw]; s->e = d->wb[jw + 1];
                if (s->e <= s->s) return -2;
                s->ncell = (long)s->ex * s->ey;
            }
    for (int a = 0; a < d->p1; ++a) {
        Sub* s = &d->sub[a];
        for (int i = s->oi0; i < s->oi1; ++i) d->colown[i] = a;
        for (int li = 0; li < s->ex; ++li) {
            int gi = imod(s->ei0 + li, nlon);
            if (d->ncolcov[gi] >= 4) return -2;
            d->colcov[4 * gi + d->ncolcov[gi]++] = a;
        }
    }
    for (int b = 0; b < d->p2; ++b) {
        Sub* s = &d->sub[b * d->p1];
        for (int j = s->oj0; j < s->oj1; ++j) d->rowown[j] = b;
        for (int lj = 0; lj < s->ey; ++lj) {
            int gj = s->ej0 + lj;
            if (d->nrowcov[gj] >= 4) return -2;
            d->rowcov[4 * gj + d->nrowcov[gj]++] = b;
        }
    }
    return 0;
}
static inline int sub_index(const DD* d, int jw, int b, int a) { return (jw * d->p2 + b) * d->p1 + a; }
/* local cell of global (gi,gj) in sub s, or -1 */
static inline long local_cell(const DD* d, const Sub* s, int gi, int gj)
{
    int li = imod(gi - s->ei0, d->m.nlon), lj = gj - s->ej0;
    if (li >= s->ex || lj < 0 || lj >= s->ey) return -1;
    return (long)lj * s->ex + li;
}
/* O6: restriction weight = 1/multiplicity (Def 4 l.170 generalised to 2-D tiles, R6) */
static inline double w_space(const DD* d, int gi, int gj)
{ return 1.0 / (double)(d->ncolcov[gi] * d->nrowcov[gj]); }
static inline int mult_time(const DD* d, int level)
{
    for (int j = 1; j < d->q; ++j) if (d->wb[j] == level) return 2;
    return 1;
}
static inline size_t gidx(const DD* d, int fl, int gj, int gi)
{ return ((size_t)fl * d->m.nlat + gj) * d->m.nlon + gi; }
static inline const double* ub_level(const DD* d, int level)
{ return d->ubtraj + (size_t)level * NF * d->m.nlat * d->m.nlon; }

/* frozen values: the neighbour's own data from the previous outer iteration; iteration 0: the
 * background trajectory (Alg 1 l.455; R14, R15) */
static inline double frozen_traj(const DD* d, int k, int level, int fl, long cell, int gi, int gj)
{
    const Sub* s = &d->sub[k];
    if (d->traj_prev[k]) return d->traj_prev[k][((size_t)(level - s->s) * NF + fl) * s->ncell + cell];
    return ub_level(d, level)[gidx(d, fl, gj, gi)];
}
static inline double frozen_ctrl(const DD* d, int k, int fl, long cell, int gi, int gj)
{
    const Sub* s = &d->sub[k];
    if (d->x_prev[k]) return d->x_prev[k][(size_t)fl * s->ncell + cell];
    return ub_level(d, s->s)[gidx(d, fl, gj, gi)];
}

/* Build the padded tile of sub k at window level `level`: interior = Zint [3][ncell]; ghost ring
 * = frozen values from the trajectory of the tile that OWNS each ghost cell, same window. */
static void fill_padded(const DD* d, int k, int level, const double* Zint, double* Zp, Region* r)
{
    const Sub* s = &d->sub[k];
    r->px = s->ex + 2 * s->gx; r->py = s->ey + s->gys + s->gyn;
    r->joff = s->ej0 - s->gys;
    r->per_x = s->gx == 0; r->wall_s = s->gys == 0; r->wall_n = s->gyn == 0;
    for (int fl = 0; fl < NF; ++fl)
        for (int pj = 0; pj < r->py; ++pj)
            for (int pi = 0; pi < r->px; ++pi) {
                int li = pi - s->gx, lj = pj - s->gys;
                double v;
                if (li >= 0 && li < s->ex && lj >= 0 && lj < s->ey)
                    v = Zint[(size_t)fl * s->ncell + (size_t)lj * s->ex + li];
                else {
                    int gi = imod(s->ei0 + li, d->m.nlon), gj = s->ej0 + lj;
                    int ko = sub_index(d, s->jw, d->rowown[gj], d->colown[gi]);
                    long c = local_cell(d, &d->sub[ko], gi, gj);
                    v = frozen_traj(d, ko, level, fl, c, gi, gj);
                }
                Zp[((size_t)fl * r->py + pj) * r->px + pi] = v;
            }
}
static void interior_to_padded(const Sub* s, const Region* r, const double* X, double* P)
{
    memset(P, 0, sizeof(double) * NF * r->px * r->py);
    for (int fl = 0; fl < NF; ++fl)
        for (int lj = 0; lj < s->ey; ++lj)
            for (int li = 0; li < s->ex; ++li)
                P[((size_t)fl * r->py + lj + s->gys) * r->px + li + s->gx] =
                    X[(size_t)fl * s->ncell + (size_t)lj * s->ex + li];
}
static void padded_to_interior(const Sub* s, const Region* r, const double* P, double* X)
{
    for (int fl = 0; fl < NF; ++fl)
        for (int lj = 0; lj < s->ey; ++lj)
            for (int li = 0; li < s->ex; ++li)
                X[(size_t)fl * s->ncell + (size_t)lj * s->ex + li] =
                    P[((size_t)fl * r->py + lj + s->gys) * r->px + li + s->gx];
}

/* ------------------------------------------------------------------ O7: J_ji and gradient -- */
typedef struct { double total, bg, obs, ov_space, ov_pred, ov_succ; } CostParts;

/* x: control = state on the extended tile at level s_j, [3][ncell], physical units.
 * traj: [(e-s+1)][3][ncell] work/output.  grad (may be NULL): dJ_ji/dx. */
static void local_eval(const DD* d, int k, const double* x, CostParts* cp, double* grad, double* traj)
{
    const Sub* s = &d->sub[k];
    const int nlon = d->m.nlon;
    const int W = s->e - s->s;
    const long nc = s->ncell;
    Region r;
    size_t np = (size_t)(s->ex + 2 * s->gx) * (s->ey + s->gys + s->gyn);
    double* Zp = malloc(sizeof(double) * NF * np);
    double* Za = calloc(NF * np, sizeof(double));
    double* Z1 = calloc(NF * np, sizeof(double));
    /* forward sweep over the window (eq (1) l.53-57 restricted, Def 6 l.210-219) */
    memcpy(traj, x, sizeof(double) * NF * nc);
    for (int n = 0; n < W; ++n) {
        fill_padded(d, k, s->s + n, traj + (size_t)n * NF * nc, Zp, &r);
        region_forward(&d->m, &r, Zp, Za, Z1);
        padded_to_interior(s, &r, Z1, traj + (size_t)(n + 1) * NF * nc);
    }
    /* cost terms, eq (25) l.338-344, squared weighted 2-norms without 1/2 (R5) */
    long double Jbg = 0, Jobs = 0, Jsp = 0, Jpred = 0, Jsucc = 0;
    const double* ubs = ub_level(d, s->s);
    const double bgw = s->jw == 0 ? 1.0 : d->bgw;      /* DESIGN.md R7 */
    for (int fl = 0; fl < NF; ++fl) {
        double ib = 1.0 / (d->sig_b[fl] * d->sig_b[fl]);
        for (int lj = 0; lj < s->ey; ++lj)
            for (int li = 0; li < s->ex; ++li) {
                int gi = imod(s->ei0 + li, nlon), gj = s->ej0 + lj;
                long c = (long)lj * s->ex + li;
                double xv = x[(size_t)fl * nc + c];
                double db = xv - ubs[gidx(d, fl, gj, gi)];
                Jbg += (long double)(bgw * w_space(d, gi, gj) * db * db * ib);              /* (25a) */
                /* (25c) case 1: every other extended tile of this window that contains the cell */
                for (int cb = 0; cb < d->nrowcov[gj]; ++cb)
                    for (int ca = 0; ca < d->ncolcov[gi]; ++ca) {
                        int a2 = d->colcov[4 * gi + ca], b2 = d->rowcov[4 * gj + cb];
                        if (a2 == s->a && b2 == s->b) continue;
                        int k2 = sub_index(d, s->jw, b2, a2);
                        long c2 = local_cell(d, &d->sub[k2], gi, gj);
                        double dv = xv - frozen_ctrl(d, k2, fl, c2, gi, gj);
                        Jsp += (long double)(dv * dv * ib);
                    }
                if (s->jw > 0) {                           /* (25c) case 2, predecessor window */
                    int kp = sub_index(d, s->jw - 1, s->b, s->a);
                    double dv = xv - frozen_traj(d, kp, s->s, fl, c, gi, gj);
                    Jpred += (long double)(dv * dv * ib);
                }
                if (s->jw < d->q - 1) {                    /* (25c) case 2, successor window */
                    int kn = sub_index(d, s->jw + 1, s->b, s->a);
                    double dv = traj[((size_t)W * NF + fl) * nc + c] - frozen_ctrl(d, kn, fl, c, gi, gj);
                    Jsucc += (long double)(dv * dv * ib);
                }
            }
    }
    if (d->ovl_levels)                                    /* (25c) case 1 on the levels n = 1 .. W as well */
        for (int n = 1; n <= W; ++n)
            for (int fl = 0; fl < NF; ++fl) {
                double ib = 1.0 / (d->sig_b[fl] * d->sig_b[fl]);
                for (int lj = 0; lj < s->ey; ++lj)
                    for (int li = 0; li < s->ex; ++li) {
                        int gi = imod(s->ei0 + li, nlon), gj = s->ej0 + lj;
                        long c = (long)lj * s->ex + li;
                        double zv = traj[((size_t)n * NF + fl) * nc + c];
                        for (int cb = 0; cb < d->nrowcov[gj]; ++cb)
                            for (int ca = 0; ca < d->ncolcov[gi]; ++ca) {
                                int a2 = d->colcov[4 * gi + ca], b2 = d->rowcov[4 * gj + cb];
                                if (a2 == s->a && b2 == s->b) continue;
                                int k2 = sub_index(d, s->jw, b2, a2);
                                long c2 = local_cell(d, &d->sub[k2], gi, gj);
                                double dv = zv - frozen_traj(d, k2, s->s + n, fl, c2, gi, gj);
                                Jsp += (long double)(dv * dv * ib);
                            }
                    }
            }
    if (d->have_obs)
        for (long q = 0; q < d->nlocobs[k]; ++q) {        /* (25b) */
            const LocObs* ob = &d->locobs[k][q];
            int level = d->olev[ob->tidx];
            int lj = (int)(ob->cell / s->ex), li = (int)(ob->cell % s->ex);
            int gi = imod(s->ei0 + li, nlon), gj = s->ej0 + lj;
            double wt = w_space(d, gi, gj) / (double)mult_time(d, level);
            double rr = traj[((size_t)(level - s->s) * NF + ob->fld) * nc + ob->cell] - ob->y;
            Jobs += (long double)(wt * rr * rr / (d->sig_o[ob->fld] * d->sig_o[ob->fld]));
        }
    cp->bg = (double)Jbg; cp->obs = (double)(d->lambda * Jobs);
    cp->ov_space = (double)(d->mu * Jsp); cp->ov_pred = (double)(d->mu * Jpred);
    cp->ov_succ = (double)(d->mu * Jsucc);
    cp->total = (double)(Jbg + d->lambda * Jobs + d->mu * (Jsp + Jpred + Jsucc));

    if (grad) {
        /* backward sweep: adjoint variable starts at the window end with the end-of-window
         * forcing, collects H^T R^-1 (misfit) at every observation level, goes through the step
         * adjoints in reverse (eq (4) l.98); perturbations of frozen ghost data are zero. */
        double* lam = calloc(NF * nc, sizeof(double));
        double* L1 = malloc(sizeof(double) * NF * np);
        double* L0 = malloc(sizeof(double) * NF * np);
        double* A = malloc(sizeof(double) * NF * np);
        double* HB = malloc(sizeof(double) * np);
        double* UB = malloc(sizeof(double) * np);
        if (s->jw < d->q - 1) {
            int kn = sub_index(d, s->jw + 1, s->b, s->a);
            for (int fl = 0; fl < NF; ++fl) {
                double ib = 1.0 / (d->sig_b[fl] * d->sig_b[fl]);
                for (int lj = 0; lj < s->ey; ++lj)
                    for (int li = 0; li < s->ex; ++li) {
                        int gi = imod(s->ei0 + li, nlon), gj = s->ej0 + lj;
                        long c = (long)lj * s->ex + li;
                        double dv = traj[((size_t)W * NF + fl) * nc + c] - frozen_ctrl(d, kn, fl, c, gi, gj);
                        lam[(size_t)fl * nc + c] += 2.0 * d->mu * dv * ib;
                    }
            }
        }
        for (int n = W; n >= 0; --n) {
            int level = s->s + n;
            if (d->have_obs)
                for (long q = 0; q < d->nlocobs[k]; ++q) {
                    const LocObs* ob = &d->locobs[k][q];
                    if (d->olev[ob->tidx] != level) continue;
                    int lj = (int)(ob->cell / s->ex), li = (int)(ob->cell % s->ex);
                    int gi = imod(s->ei0 + li, nlon), gj = s->ej0 + lj;
                    double wt = w_space(d, gi, gj) / (double)mult_time(d, level);
                    double rr = traj[((size_t)n * NF + ob->fld) * nc + ob->cell] - ob->y;
                    lam[(size_t)ob->fld * nc + ob->cell] +=
                        2.0 * d->lambda * wt * rr / (d->sig_o[ob->fld] * d->sig_o[ob->fld]);
                }
            if (d->ovl_levels && n > 0)                    /* forcing of the all-level overlap term */
                for (int fl = 0; fl < NF; ++fl) {
                    double ib = 1.0 / (d->sig_b[fl] * d->sig_b[fl]);
                    for (int lj = 0; lj < s->ey; ++lj)
                        for (int li = 0; li < s->ex; ++li) {
                            int gi = imod(s->ei0 + li, nlon), gj = s->ej0 + lj;
                            long c = (long)lj * s->ex + li;
                            double zv = traj[((size_t)n * NF + fl) * nc + c];
                            for (int cb = 0; cb < d->nrowcov[gj]; ++cb)
                                for (int ca = 0; ca < d->ncolcov[gi]; ++ca) {
                                    int a2 = d->colcov[4 * gi + ca], b2 = d->rowcov[4 * gj + cb];
                                    if (a2 == s->a && b2 == s->b) continue;
                                    int k2 = sub_index(d, s->jw, b2, a2);
                                    long c2 = local_cell(d, &d->sub[k2], gi, gj);
                                    lam[(size_t)fl * nc + c] += 2.0 * d->mu * (zv - frozen_traj(d, k2, level, fl, c2, gi, gj)) * ib;
                                }
                        }
                }
            if (n > 0) {
                fill_padded(d, k, level - 1, traj + (size_t)(n - 1) * NF * nc, Zp, &r);
                region_forward(&d->m, &r, Zp, Za, Z1);
                interior_to_padded(s, &r, lam, L1);
                region_adjoint(&d->m, &r, Zp, Za, Z1, L1, A, HB, UB, L0);
                padded_to_interior(s, &r, L0, lam);       /* contributions to ghost cells dropped */
            }
        }
        for (int fl = 0; fl < NF; ++fl) {
            double ib = 1.0 / (d->sig_b[fl] * d->sig_b[fl]);
            for (int lj = 0; lj < s->ey; ++lj)
                for (int li = 0; li < s->ex; ++li) {
                    int gi = imod(s->ei0 + li, nlon), gj = s->ej0 + lj;
                    long c = (long)lj * s->ex + li;
                    double xv = x[(size_t)fl * nc + c];
                    double gsum = lam[(size_t)fl * nc + c];
                    gsum += 2.0 * (s->jw == 0 ? 1.0 : d->bgw) * w_space(d, gi, gj) * (xv - ubs[gidx(d, fl, gj, gi)]) * ib;
                    for (int cb = 0; cb < d->nrowcov[gj]; ++cb)
                        for (int ca = 0; ca < d->ncolcov[gi]; ++ca) {
                            int a2 = d->colcov[4 * gi + ca], b2 = d->rowcov[4 * gj + cb];
                            if (a2 == s->a && b2 == s->b) continue;
                            int k2 = sub_index(d, s->jw, b2, a2);
                            long c2 = local_cell(d, &d->sub[k2], gi, gj);
                            gsum += 2.0 * d->mu * (xv - frozen_ctrl(d, k2, fl, c2, gi, gj)) * ib;
                        }
                    if (s->jw > 0) {
                        int kp = sub_index(d, s->jw - 1, s->b, s->a);
                        gsum += 2.0 * d->mu * (xv - frozen_traj(d, kp, s->s, fl, c, gi, gj)) * ib;
                    }
                    grad[(size_t)fl * nc + c] = gsum;
                }
        }
        free(lam); free(L1); free(L0); free(A); free(HB); free(UB);
    }
    free(Zp); free(Za); free(Z1);
}

/* ------------------------------------------------------------------ O4: global J, gradient - */
static void global_forward(const DD* d, const double* x0, int nsteps, double* traj /*[(nsteps+1)]*/)
{
    Region r = { d->m.nlon, d->m.nlat, 0, 1, 1, 1 };
    size_t n3 = (size_t)NF * d->m.nlon * d->m.nlat;
    double* Za = malloc(sizeof(double) * n3);
    memcpy(traj, x0, sizeof(double) * n3);
    for (int n = 0; n < nsteps; ++n)
        region_forward(&d->m, &r, traj + (size_t)n * n3, Za, traj + (size_t)(n + 1) * n3);
    free(Za);
}
/* J(x) = ||x - x_b||^2_{B^-1} + lambda sum_k ||H_k(M(x)) - v_k||^2_{R^-1}, eq (6) l.111 */
static double global_eval(const DD* d, const double* x, double* grad, double* parts /*[2] or NULL*/)
{
    const int nlon = d->m.nlon, nlat = d->m.nlat, N = d->nsteps;
    size_t n1 = (size_t)nlon * nlat, n3 = NF * n1;
    Region r = { nlon, nlat, 0, 1, 1, 1 };
    double* traj = malloc(sizeof(double) * n3 * (N + 1));
    global_forward(d, x, N, traj);
    long double Jb = 0, Jo = 0;
    for (int fl = 0; fl < NF; ++fl) {
        double ib = 1.0 / (d->sig_b[fl] * d->sig_b[fl]);
        for (size_t c = 0; c < n1; ++c) {
            double db = x[fl * n1 + c] - d->xb[fl * n1 + c];
            Jb += (long double)(db * db * ib);
        }
    }
    if (d->have_obs)
        for (int tk = 0; tk < d->ntimes; ++tk) {
            const double* Z = traj + (size_t)d->olev[tk] * n3;
            for (long long q = d->ooff[tk]; q < d->ooff[tk + 1]; ++q) {
                int fl = (int)(d->oidx[q] / (long)n1);
                double rr = Z[d->oidx[q]] - d->oval[q];
                Jo += (long double)(rr * rr / (d->sig_o[fl] * d->sig_o[fl]));
            }
        }
    if (parts) { parts[0] = (double)Jb; parts[1] = (double)(d->lambda * Jo); }
    if (grad) {
        double* lam = calloc(n3, sizeof(double));
        double* Za = malloc(sizeof(double) * n3); double* Z1 = malloc(sizeof(double) * n3);
        double* L0 = malloc(sizeof(double) * n3); double* A = malloc(sizeof(double) * n3);
        double* HB = malloc(sizeof(double) * n1); double* UB = malloc(sizeof(double) * n1);
        int tk = d->have_obs ? d->ntimes - 1 : -1;
        for (int n = N; n >= 0; --n) {
            while (tk >= 0 && d->olev[tk] > n) --tk;
            if (tk >= 0 && d->olev[tk] == n) {
                const double* Z = traj + (size_t)n * n3;
                for (long long q = d->ooff[tk]; q < d->ooff[tk + 1]; ++q) {
                    int fl = (int)(d->oidx[q] / (long)n1);
                    lam[d->oidx[q]] += 2.0 * d->lambda * (Z[d->oidx[q]] - d->oval[q])
                                       / (d->sig_o[fl] * d->sig_o[fl]);
                }
            }
            if (n > 0) {
                const double* Z0 = traj + (size_t)(n - 1) * n3;
                region_forward(&d->m, &r, Z0, Za, Z1);
                region_adjoint(&d->m, &r, Z0, Za, Z1, lam, A, HB, UB, L0);
                memcpy(lam, L0, sizeof(double) * n3);
            }
        }
        for (int fl = 0; fl < NF; ++fl) {
            double ib = 1.0 / (d->sig_b[fl] * d->sig_b[fl]);
            for (size_t c = 0; c < n1; ++c)
                grad[fl * n1 + c] = lam[fl * n1 + c] + 2.0 * (x[fl * n1 + c] - d->xb[fl * n1 + c]) * ib;
        }
        free(lam); free(Za); free(Z1); free(L0); free(A); free(HB); free(UB);
    }
    free(traj);
    return (double)(Jb + d->lambda * Jo);
}

/* ------------------------------------------------------------------ O8: L-BFGS ------------
 * Liu-Nocedal two-loop recursion (PAPER.md ref [29], l.941, Remark 3 l.595) with the constants
 * of DESIGN.md R10: exactly n_iter iterations; H0 = (s'y / y'y) I; first iteration (or empty
 * history) d = -g with trial step 1/||g||; Armijo backtracking c1, halving, trials t0/2^b for
 * b = 0..max_bt; no acceptable trial: keep the point, clear the history; pair skipped when
 * s'y <= 1e-12 ||s|| ||y||.  fn(ctx, w, want_grad, &J, g). */
typedef void (*orc_evalfn)(void* ctx, const double* w, int want_grad, double* J, double* g);

static long double ldot(const double* a, const double* b, long n)
{ long double s = 0; for (long i = 0; i < n; ++i) s += (long double)(a[i] * b[i]); return s; }

static double lbfgs_run(long n, int m, int n_iter, int max_bt, double c1, orc_evalfn fn, void* ctx,
                        double* w, double* Jfirst)
{
    double *g = malloc(sizeof(double) * n), *gn = malloc(sizeof(double) * n);
    double *dvec = malloc(sizeof(double) * n), *wt = malloc(sizeof(double) * n);
    double *S = malloc(sizeof(double) * n * (m > 0 ? m : 1)), *Y = malloc(sizeof(double) * n * (m > 0 ? m : 1));
    double *rho = malloc(sizeof(double) * (m > 0 ? m : 1)), *alpha = malloc(sizeof(double) * (m > 0 ? m : 1));
    int nh = 0;                                  /* pairs stored, oldest first */
    double J;
    fn(ctx, w, 1, &J, g);
    if (Jfirst) *Jfirst = J;
    for (int it = 0; it < n_iter; ++it) {
        double gnorm = sqrt((double)ldot(g, g, n));
        if (!(gnorm > 0.0)) break;
        double t0, gd;
        if (nh > 0) {
            memcpy(dvec, g, sizeof(double) * n);
            for (int i = nh - 1; i >= 0; --i) {
                alpha[i] = rho[i] * (double)ldot(S + (size_t)i * n, dvec, n);
                for (long c = 0; c < n; ++c) dvec[c] -= alpha[i] * Y[(size_t)i * n + c];
            }
            const double* sl = S + (size_t)(nh - 1) * n; const double* yl = Y + (size_t)(nh - 1) * n;
            double gamma = (double)(ldot(sl, yl, n) / ldot(yl, yl, n));
            for (long c = 0; c < n; ++c) dvec[c] *= gamma;
            for (int i = 0; i < nh; ++i) {
                double beta = rho[i] * (double)ldot(Y + (size_t)i * n, dvec, n);
                for (long c = 0; c < n; ++c) dvec[c] += S[(size_t)i * n + c] * (alpha[i] - beta);
            }
            for (long c = 0; c < n; ++c) dvec[c] = -dvec[c];
            t0 = 1.0;
            gd = (double)ldot(g, dvec, n);
            if (!(gd < 0.0)) nh = 0;             /* not a descent direction: restart */
        }
        if (nh == 0) {
            for (long c = 0; c < n; ++c) dvec[c] = -g[c];
            t0 = 1.0 / gnorm;
            gd = -(gnorm * gnorm);
        }
        double t = t0, Jt = 0.0; int ok = 0;
        for (int b = 0; b <= max_bt; ++b) {
            for (long c = 0; c < n; ++c) wt[c] = w[c] + t * dvec[c];
            fn(ctx, wt, 0, &Jt, NULL);
            if (Jt <= J + c1 * t * gd) { ok = 1; break; }
            t *= 0.5;
        }
        if (!ok) { nh = 0; continue; }
        fn(ctx, wt, 1, &Jt, gn);
        if (m > 0) {
            if (nh == m) {                       /* drop the oldest pair */
                memmove(S, S + n, sizeof(double) * n * (m - 1));
                memmove(Y, Y + n, sizeof(double) * n * (m - 1));
                memmove(rho, rho + 1, sizeof(double) * (m - 1));
                nh = m - 1;
            }
            double* sn = S + (size_t)nh * n; double* yn = Y + (size_t)nh * n;
            for (long c = 0; c < n; ++c) { sn[c] = wt[c] - w[c]; yn[c] = gn[c] - g[c]; }
            double sy = (double)ldot(sn, yn, n);
            double ss = sqrt((double)ldot(sn, sn, n)), yy = sqrt((double)ldot(yn, yn, n));
            if (sy > 1e-12 * ss * yy) { rho[nh] = 1.0 / sy; ++nh; }
        }
        memcpy(w, wt, sizeof(double) * n);
        memcpy(g, gn, sizeof(double) * n);
        J = Jt;
    }
    free(g); free(gn); free(dvec); free(wt); free(S); free(Y); free(rho); free(alpha);
    return J;
}

/* local functional in the B-preconditioned variable w = (x - u^b(s_j))/sigma_b, eq (44) l.630 */
typedef struct { const DD* d; int k; double* x; double* gx; double* traj; } LocCtx;
static void w_to_x(const DD* d, int k, const double* w, double* x)
{
    const Sub* s = &d->sub[k];
    const double* ubs = ub_level(d, s->s);
    for (int fl = 0; fl < NF; ++fl)
        for (int lj = 0; lj < s->ey; ++lj)
            for (int li = 0; li < s->ex; ++li) {
                int gi = imod(s->ei0 + li, d->m.nlon), gj = s->ej0 + lj;
                size_t c = (size_t)fl * s->ncell + (size_t)lj * s->ex + li;
                x[c] = ubs[gidx(d, fl, gj, gi)] + d->sig_b[fl] * w[c];
            }
}
static void local_fn(void* ctx, const double* w, int want_grad, double* J, double* g)
{
    LocCtx* c = ctx; const Sub* s = &c->d->sub[c->k];
    CostParts cp;
    w_to_x(c->d, c->k, w, c->x);
    local_eval(c->d, c->k, c->x, &cp, want_grad ? c->gx : NULL, c->traj);
    *J = cp.total;
    if (want_grad)
        for (int fl = 0; fl < NF; ++fl)
            for (long q = 0; q < s->ncell; ++q)
                g[fl * s->ncell + q] = c->d->sig_b[fl] * c->gx[fl * s->ncell + q];
}

/* ================================================================== C interface ========== */
void* orc_create(int nlon, int nlat, double radius, double omega, double gravity, double cos_clamp,
                 double diffusion, int p_lon, int p_lat, int q_time, int overlap, double mu,
                 double lambda, double dt, int nsteps, int lbfgs_m, int n_inner, int max_bt,
                 double c1, int* status)
{
    DD* d = calloc(1, sizeof(DD));
    d->m.nlon = nlon; d->m.nlat = nlat; d->m.a = radius; d->m.Omega = omega; d->m.g = gravity;
    d->m.cos_clamp = cos_clamp; d->m.kappa = diffusion; d->m.dt = dt;
    d->nsteps = nsteps; d->p1 = p_lon; d->p2 = p_lat; d->q = q_time; d->o = overlap;
    d->mu = mu; d->lambda = lambda; d->bgw = 0.0; d->ovl_levels = 0;
    d->lbfgs_m = lbfgs_m; d->n_inner = n_inner; d->max_bt = max_bt; d->c1 = c1;
    if (nlon < 3 || nlat < 2 || nsteps < 1) { *status = -1; free(d); return NULL; }
    model_tables(&d->m);
    int rc = build_decomposition(d);
    if (rc) { *status = rc; return NULL; }
    d->w_prev = calloc(d->nsub, sizeof(double*)); d->x_prev = calloc(d->nsub, sizeof(double*));
    d->traj_prev = calloc(d->nsub, sizeof(double*));
    d->w_cur = calloc(d->nsub, sizeof(double*)); d->x_cur = calloc(d->nsub, sizeof(double*));
    d->traj_cur = calloc(d->nsub, sizeof(double*));
    *status = 0;
    return d;
}
/* weight of the background term (25a) in the windows j > 0 (R7: default 0; 1 = as printed) */
void orc_set_bg_weight(void* h, double w) { ((DD*)h)->bgw = w; }
void orc_set_overlap_levels(void* h, int on) { ((DD*)h)->ovl_levels = on != 0; }
static void free_local(DD* d)
{
    for (int k = 0; k < d->nsub; ++k) {
        free(d->w_prev[k]); free(d->x_prev[k]); free(d->traj_prev[k]);
        free(d->w_cur[k]); free(d->x_cur[k]); free(d->traj_cur[k]);
        d->w_prev[k] = d->x_prev[k] = d->traj_prev[k] = NULL;
        d->w_cur[k] = d->x_cur[k] = d->traj_cur[k] = NULL;
    }
}
void orc_destroy(void* h)
{
    DD* d = h; if (!d) return;
    free_local(d);
    if (d->locobs) { for (int k = 0; k < d->nsub; ++k) free(d->locobs[k]); free(d->locobs); free(d->nlocobs); }
    free(d->olev); free(d->ooff); free(d->oidx); free(d->oval);
    free(d->xb); free(d->ubtraj); free(d->sub); free(d->colown); free(d->rowown);
    free(d->ncolcov); free(d->colcov); free(d->nrowcov); free(d->rowcov); free(d->wb);
    free(d->w_prev); free(d->x_prev); free(d->traj_prev); free(d->w_cur); free(d->x_cur); free(d->traj_cur);
    model_free(&d->m); free(d);
}
int orc_nsub(void* h) { return ((DD*)h)->nsub; }
/* out: a,b,jw, oi0,oi1,oj0,oj1, ei0,ej0,ex,ey, gx,gys,gyn, s,e */
void orc_sub_info(void* h, int k, int* out)
{
    Sub* s = &((DD*)h)->sub[k];
    int v[16] = { s->a, s->b, s->jw, s->oi0, s->oi1, s->oj0, s->oj1, s->ei0, s->ej0, s->ex, s->ey,
                  s->gx, s->gys, s->gyn, s->s, s->e };
    memcpy(out, v, sizeof(v));
}
/* row tables f,t,cz,rp,rm,mc (each nlat) and cm: for the closed-form pins */
void orc_row_tables(void* h, double* out6, double* cm)
{
    DD* d = h; int n = d->m.nlat;
    memcpy(out6, d->m.f, sizeof(double) * n); memcpy(out6 + n, d->m.t, sizeof(double) * n);
    memcpy(out6 + 2 * n, d->m.cz, sizeof(double) * n); memcpy(out6 + 3 * n, d->m.rp, sizeof(double) * n);
    memcpy(out6 + 4 * n, d->m.rm, sizeof(double) * n); memcpy(out6 + 5 * n, d->m.mc, sizeof(double) * n);
    *cm = d->m.cm;
}
/* restriction weight of sub k at `level` on its extended tile (0 if level outside its window) */
void orc_sub_weight(void* h, int k, int level, double* out)
{
    DD* d = h; Sub* s = &d->sub[k];
    for (int lj = 0; lj < s->ey; ++lj)
        for (int li = 0; li < s->ex; ++li) {
            int gi = imod(s->ei0 + li, d->m.nlon), gj = s->ej0 + lj;
            out[(size_t)lj * s->ex + li] =
                (level < s->s || level > s->e) ? 0.0 : w_space(d, gi, gj) / mult_time(d, level);
        }
}
/* global model: one step, its TLM and its adjoint (all [3][nlat][nlon]) */
void orc_step(void* h, const double* Z0, double* Z1)
{
    DD* d = h; Region r = { d->m.nlon, d->m.nlat, 0, 1, 1, 1 };
    double* Za = malloc(sizeof(double) * NF * r.px * r.py);
    region_forward(&d->m, &r, Z0, Za, Z1); free(Za);
}
void orc_step_tlm(void* h, const double* Z0, const double* dZ0, double* dZ1)
{
    DD* d = h; Region r = { d->m.nlon, d->m.nlat, 0, 1, 1, 1 };
    size_t n3 = (size_t)NF * r.px * r.py;
    double *Za = malloc(sizeof(double) * n3), *Z1 = malloc(sizeof(double) * n3), *dZa = malloc(sizeof(double) * n3);
    region_forward(&d->m, &r, Z0, Za, Z1);
    region_tlm(&d->m, &r, Z0, Za, Z1, dZ0, dZa, dZ1);
    free(Za); free(Z1); free(dZa);
}
void orc_step_adj(void* h, const double* Z0, const double* L1, double* L0)
{
    DD* d = h; Region r = { d->m.nlon, d->m.nlat, 0, 1, 1, 1 };
    size_t n1 = (size_t)r.px * r.py, n3 = NF * n1;
    double *Za = malloc(sizeof(double) * n3), *Z1 = malloc(sizeof(double) * n3), *A = malloc(sizeof(double) * n3);
    double *HB = malloc(sizeof(double) * n1), *UB = malloc(sizeof(double) * n1);
    region_forward(&d->m, &r, Z0, Za, Z1);
    region_adjoint(&d->m, &r, Z0, Za, Z1, L1, A, HB, UB, L0);
    free(Za); free(Z1); free(A); free(HB); free(UB);
}
/* run the global model from x0 and return the states at the given ascending levels */
void orc_forecast(void* h, const double* x0, int nlev, const int* levels, double* out)
{
    DD* d = h; Region r = { d->m.nlon, d->m.nlat, 0, 1, 1, 1 };
    size_t n3 = (size_t)NF * r.px * r.py;
    double *Z = malloc(sizeof(double) * n3), *Zn = malloc(sizeof(double) * n3), *Za = malloc(sizeof(double) * n3);
    memcpy(Z, x0, sizeof(double) * n3);
    int q = 0, last = nlev > 0 ? levels[nlev - 1] : 0;
    for (int n = 0; n <= last; ++n) {
        while (q < nlev && levels[q] == n) { memcpy(out + (size_t)q * n3, Z, sizeof(double) * n3); ++q; }
        if (n < last) { region_forward(&d->m, &r, Z, Za, Zn); double* t = Z; Z = Zn; Zn = t; }
    }
    free(Z); free(Zn); free(Za);
}
/* Alg 1 l.452: u^b = M(u_0^b); l.455: u_ji^0 = u_ji^b.  Frozen data := background (NULL). */
int orc_set_background(void* h, const double* xb, const double* sigma_b)
{
    DD* d = h; size_t n3 = (size_t)NF * d->m.nlon * d->m.nlat;
    for (int f = 0; f < NF; ++f) { if (!(sigma_b[f] > 0)) return -1; d->sig_b[f] = sigma_b[f]; }
    free(d->xb); free(d->ubtraj);
    d->xb = malloc(sizeof(double) * n3); memcpy(d->xb, xb, sizeof(double) * n3);
    d->ubtraj = malloc(sizeof(double) * n3 * (d->nsteps + 1));
    if (!d->ubtraj) return -4;
    global_forward(d, xb, d->nsteps, d->ubtraj);
    free_local(d);
    d->have_bg = 1;
    return 0;
}
int orc_set_observations(void* h, int ntimes, const int* levels, const long long* offs,
                         const int* idx, const double* val, const double* sigma_o)
{
    DD* d = h; const int nlon = d->m.nlon, nlat = d->m.nlat; long n1 = (long)nlon * nlat;
    for (int f = 0; f < NF; ++f) { if (!(sigma_o[f] > 0)) return -1; d->sig_o[f] = sigma_o[f]; }
    for (int t = 0; t < ntimes; ++t) {
        if (levels[t] < 0 || levels[t] > d->nsteps || (t && levels[t] <= levels[t - 1])) return -1;
        for (long long q = offs[t]; q < offs[t + 1]; ++q) if (idx[q] < 0 || idx[q] >= NF * n1) return -1;
    }
    free(d->olev); free(d->ooff); free(d->oidx); free(d->oval);
    long long tot = ntimes ? offs[ntimes] : 0;
    d->ntimes = ntimes;
    d->olev = malloc(sizeof(int) * (ntimes + 1)); memcpy(d->olev, levels, sizeof(int) * ntimes);
    d->ooff = malloc(sizeof(long long) * (ntimes + 1)); memcpy(d->ooff, offs, sizeof(long long) * (ntimes + 1));
    d->oidx = malloc(sizeof(int) * (tot + 1)); memcpy(d->oidx, idx, sizeof(int) * tot);
    d->oval = malloc(sizeof(double) * (tot + 1)); memcpy(d->oval, val, sizeof(double) * tot);
    if (d->locobs) { for (int k = 0; k < d->nsub; ++k) free(d->locobs[k]); free(d->locobs); free(d->nlocobs); }
    d->locobs = calloc(d->nsub, sizeof(LocObs*)); d->nlocobs = calloc(d->nsub, sizeof(long));
    /* Def 8 l.239: restriction of H^(k) to Delta_j x Omega_i = the observations inside it */
    for (int pass = 0; pass < 2; ++pass) {
        if (pass) for (int k = 0; k < d->nsub; ++k) { d->locobs[k] = malloc(sizeof(LocObs) * (d->nlocobs[k] + 1)); d->nlocobs[k] = 0; }
        for (int t = 0; t < ntimes; ++t)
            for (long long q = offs[t]; q < offs[t + 1]; ++q) {
                int fl = (int)(idx[q] / n1); long c = idx[q] % n1; int gj = (int)(c / nlon), gi = (int)(c % nlon);
                for (int jw = 0; jw < d->q; ++jw) {
                    if (levels[t] < d->wb[jw] || levels[t] > d->wb[jw + 1]) continue;
                    for (int cb = 0; cb < d->nrowcov[gj]; ++cb)
                        for (int ca = 0; ca < d->ncolcov[gi]; ++ca) {
                            int k = sub_index(d, jw, d->rowcov[4 * gj + cb], d->colcov[4 * gi + ca]);
                            if (pass) {
                                LocObs* ob = &d->locobs[k][d->nlocobs[k]];
                                ob->tidx = t; ob->fld = fl; ob->cell = local_cell(d, &d->sub[k], gi, gj); ob->y = val[q];
                            }
                            d->nlocobs[k]++;
                        }
                }
            }
    }
    d->have_obs = 1;
    return 0;
}
int orc_eval_global(void* h, const double* x0, double* cost, double* grad, double* parts)
{
    DD* d = h; if (!d->have_bg) return -3;
    *cost = global_eval(d, x0, grad, parts);
    return 0;
}
/* J_ji and dJ_ji/dx of ONE subdomain at control x (physical units), with the current frozen
 * data.  parts: total,bg,obs,ov_space,ov_pred,ov_succ.  traj_out may be NULL. */
int orc_eval_local_one(void* h, int k, const double* x, double* parts, double* grad, double* traj_out)
{
    DD* d = h; if (!d->have_bg) return -3;
    Sub* s = &d->sub[k];
    double* traj = traj_out ? traj_out : malloc(sizeof(double) * NF * s->ncell * (s->e - s->s + 1));
    CostParts cp;
    local_eval(d, k, x, &cp, grad, traj);
    parts[0] = cp.total; parts[1] = cp.bg; parts[2] = cp.obs; parts[3] = cp.ov_space;
    parts[4] = cp.ov_pred; parts[5] = cp.ov_succ;
    if (!traj_out) free(traj);
    return 0;
}
/* current control (physical) of sub k: the frozen one from the last finished outer iteration */
void orc_get_control(void* h, int k, double* out)
{
    DD* d = h; Sub* s = &d->sub[k];
    if (d->x_prev[k]) { memcpy(out, d->x_prev[k], sizeof(double) * NF * s->ncell); return; }
    double* w0 = calloc(NF * s->ncell, sizeof(double));
    w_to_x(d, k, w0, out); free(w0);
}
/* gathered state at `level`: weighted extension-sum, eq (12)-(13) l.194-201 (R11) */
void orc_get_trajectory(void* h, int level, double* out)
{
    DD* d = h; size_t n3 = (size_t)NF * d->m.nlon * d->m.nlat;
    memset(out, 0, sizeof(double) * n3);
    for (int k = 0; k < d->nsub; ++k) {
        Sub* s = &d->sub[k];
        if (level < s->s || level > s->e) continue;
        for (int fl = 0; fl < NF; ++fl)
            for (int lj = 0; lj < s->ey; ++lj)
                for (int li = 0; li < s->ex; ++li) {
                    int gi = imod(s->ei0 + li, d->m.nlon), gj = s->ej0 + lj;
                    long c = (long)lj * s->ex + li;
                    double wt = w_space(d, gi, gj) / mult_time(d, level);
                    out[gidx(d, fl, gj, gi)] += wt * frozen_traj(d, k, level, fl, c, gi, gj);
                }
    }
}
static void gather_analysis(const DD* d, double* out)
{
    size_t n3 = (size_t)NF * d->m.nlon * d->m.nlat;
    memset(out, 0, sizeof(double) * n3);
    for (int k = 0; k < d->p1 * d->p2; ++k) {          /* window 0 */
        const Sub* s = &d->sub[k];
        for (int fl = 0; fl < NF; ++fl)
            for (int lj = 0; lj < s->ey; ++lj)
                for (int li = 0; li < s->ex; ++li) {
                    int gi = imod(s->ei0 + li, d->m.nlon), gj = s->ej0 + lj;
                    long c = (long)lj * s->ex + li;
                    out[gidx(d, fl, gj, gi)] += w_space(d, gi, gj) * frozen_ctrl(d, k, fl, c, gi, gj);
                }
    }
}
/* O9: Algorithm 1 l.443-472, additive (Jacobi) outer iteration (R16), exactly outer_iters
 * iterations (R17).  history[(outer_iters+1)][3] = J(gathered analysis), sum_ji J_ji, delta_l. */
static double gn_run(const DD* d, int k, int n_gn, int n_cg, double* w, double* x, double* gx, double* traj,
                     double* J0);
static int run_impl(void* h, int outer_iters, double* analysis, double* history, int gn, int n_gn, int n_cg)
{
    DD* d = h; if (!d->have_bg) return -3;
    size_t n3 = (size_t)NF * d->m.nlon * d->m.nlat;
    double* Jfirst = malloc(sizeof(double) * d->nsub);
    double* Jlast = malloc(sizeof(double) * d->nsub);
    double* dmax = malloc(sizeof(double) * d->nsub);
    double* xa = malloc(sizeof(double) * n3);
    gather_analysis(d, xa);
    history[0] = global_eval(d, xa, NULL, NULL); history[1] = 0.0; history[2] = 0.0;
    if (outer_iters == 0) {
        long double sj = 0;
        for (int k = 0; k < d->nsub; ++k) {
            Sub* s = &d->sub[k]; double parts[6];
            double* x = malloc(sizeof(double) * NF * s->ncell);
            orc_get_control(d, k, x); orc_eval_local_one(d, k, x, parts, NULL, NULL); sj += parts[0]; free(x);
        }
        history[1] = (double)sj;
    }
    for (int l = 1; l <= outer_iters; ++l) {
#pragma omp parallel for schedule(dynamic)
        for (int k = 0; k < d->nsub; ++k) {
            Sub* s = &d->sub[k]; long n = NF * s->ncell; int W = s->e - s->s;
            d->w_cur[k] = malloc(sizeof(double) * n); d->x_cur[k] = malloc(sizeof(double) * n);
            d->traj_cur[k] = malloc(sizeof(double) * n * (W + 1));
            if (d->w_prev[k]) memcpy(d->w_cur[k], d->w_prev[k], sizeof(double) * n);
            else memset(d->w_cur[k], 0, sizeof(double) * n);
            LocCtx c = { d, k, malloc(sizeof(double) * n), malloc(sizeof(double) * n), d->traj_cur[k] };
            if (gn) Jlast[k] = gn_run(d, k, n_gn, n_cg, d->w_cur[k], c.x, c.gx, d->traj_cur[k], &Jfirst[k]);
            else Jlast[k] = lbfgs_run(n, d->lbfgs_m, d->n_inner, d->max_bt, d->c1, local_fn, &c, d->w_cur[k], &Jfirst[k]);
            /* one more forward sweep so that the stored trajectory belongs to the accepted iterate */
            CostParts cp;
            w_to_x(d, k, d->w_cur[k], d->x_cur[k]);
            local_eval(d, k, d->x_cur[k], &cp, NULL, d->traj_cur[k]);
            double* xo = malloc(sizeof(double) * n); orc_get_control(d, k, xo);
            double mx = 0; for (long q = 0; q < n; ++q) { double a = fabs(d->x_cur[k][q] - xo[q]); if (a > mx) mx = a; }
            dmax[k] = mx;
            free(xo); free(c.x); free(c.gx);
        }
        /* exchange (l.465): this iteration's results become the next one's frozen data */
        long double sj = 0, sj0 = 0; double dl = 0;
        for (int k = 0; k < d->nsub; ++k) {
            free(d->w_prev[k]); free(d->x_prev[k]); free(d->traj_prev[k]);
            d->w_prev[k] = d->w_cur[k]; d->x_prev[k] = d->x_cur[k]; d->traj_prev[k] = d->traj_cur[k];
            d->w_cur[k] = d->x_cur[k] = d->traj_cur[k] = NULL;
            sj += Jlast[k]; sj0 += Jfirst[k]; if (dmax[k] > dl) dl = dmax[k];
        }
        if (l == 1) history[1] = (double)sj0;
        gather_analysis(d, xa);
        history[3 * l] = global_eval(d, xa, NULL, NULL); history[3 * l + 1] = (double)sj; history[3 * l + 2] = dl;
    }
    gather_analysis(d, xa);
    memcpy(analysis, xa, sizeof(double) * n3);
    free(Jfirst); free(Jlast); free(dmax); free(xa);
    return 0;
}
int orc_run(void* h, int outer_iters, double* analysis, double* history)
{
    return run_impl(h, outer_iters, analysis, history, 0, 0, 0);
}

/* ------------------------------------------------------------------ O11: Gauss-Newton ------
 * The paper's own local minimiser: incremental Gauss-Newton, Algorithm 5 l.568-589 and
 * Algorithm 6 l.655-685.  J_ji = |F_ji|^2 with F_ji the stacked residuals of eq (25) l.338-344 (R5: no 1/2);
 * one Gauss-Newton iteration linearises the model about the current trajectory (TLM, Alg 6 l.14-16) and solves
 * the normal equations (42)-(43) l.620-626
 *        (grad F^T grad F) dw = - grad F^T F             <=>   H_GN dw = - grad J,   H_GN = 2 grad F^T grad F
 * in the variable w = V^+ (u - u^b), V = diag(sigma_b) (eq (44)-(46) l.630-649: the "B-preconditioned" system
 * I + (G V)^T R^-1 G V of Algorithm 7 l.688-696; here with the weights and the overlap terms of eq (25)),
 * by n_cg iterations of conjugate gradients from dw = 0 (READING, R21: Algorithm 7 names the Lanczos
 * form of [24]; CG builds the same Krylov iterates; the iteration count is fixed, no residual test), then
 * u <- u + V dw (Alg 5 l.8: full step, no line search).
 *
 * H_GN p for p in w-space: dx = V p; TLM sweep dZ^{n+1} = M_n dZ^n over the window (ghost ring frozen: zero
 * perturbation); adjoint sweep (ADJ, Alg 6 l.17-19) of the weighted TLM misfits; control-level terms. */
static void local_gn_hessvec(const DD* d, int k, const double* traj, const double* p, double* out)
{
    const Sub* s = &d->sub[k];
    const int nlon = d->m.nlon, W = s->e - s->s;
    const long nc = s->ncell;
    Region r;
    size_t np = (size_t)(s->ex + 2 * s->gx) * (s->ey + s->gys + s->gyn);
    double* Zp = malloc(sizeof(double) * NF * np);
    double* Za = calloc(NF * np, sizeof(double));
    double* Z1 = calloc(NF * np, sizeof(double));
    double* dZp = malloc(sizeof(double) * NF * np);
    double* dZa = calloc(NF * np, sizeof(double));
    double* dZ1 = calloc(NF * np, sizeof(double));
    double* dtr = malloc(sizeof(double) * NF * nc * (W + 1));          /* TLM trajectory */
    for (int fl = 0; fl < NF; ++fl)
        for (long c = 0; c < nc; ++c) dtr[(size_t)fl * nc + c] = d->sig_b[fl] * p[(size_t)fl * nc + c];
    for (int n = 0; n < W; ++n) {
        fill_padded(d, k, s->s + n, traj + (size_t)n * NF * nc, Zp, &r);
        region_forward(&d->m, &r, Zp, Za, Z1);
        interior_to_padded(s, &r, dtr + (size_t)n * NF * nc, dZp);      /* frozen ghost ring: dZ = 0 */
        memset(dZa, 0, sizeof(double) * NF * np); memset(dZ1, 0, sizeof(double) * NF * np);
        region_tlm(&d->m, &r, Zp, Za, Z1, dZp, dZa, dZ1);
        padded_to_interior(s, &r, dZ1, dtr + (size_t)(n + 1) * NF * nc);
    }
    double* lam = calloc(NF * nc, sizeof(double));
    double* L1 = malloc(sizeof(double) * NF * np);
    double* L0 = malloc(sizeof(double) * NF * np);
    double* A = malloc(sizeof(double) * NF * np);
    double* HB = malloc(sizeof(double) * np);
    double* UB = malloc(sizeof(double) * np);
    if (s->jw < d->q - 1)                                 /* (25c) successor window: 2 mu dZ^W / sigma_b^2 */
        for (int fl = 0; fl < NF; ++fl) {
            double ib = 1.0 / (d->sig_b[fl] * d->sig_b[fl]);
            for (long c = 0; c < nc; ++c)
                lam[(size_t)fl * nc + c] += 2.0 * d->mu * dtr[((size_t)W * NF + fl) * nc + c] * ib;
        }
    for (int n = W; n >= 0; --n) {
        int level = s->s + n;
        if (d->have_obs)
            for (long q = 0; q < d->nlocobs[k]; ++q) {    /* (25b): 2 lambda w H^T R^-1 H dZ^n */
                const LocObs* ob = &d->locobs[k][q];
                if (d->olev[ob->tidx] != level) continue;
                int lj = (int)(ob->cell / s->ex), li = (int)(ob->cell % s->ex);
                int gi = imod(s->ei0 + li, nlon), gj = s->ej0 + lj;
                double wt = w_space(d, gi, gj) / (double)mult_time(d, level);
                double dz = dtr[((size_t)n * NF + ob->fld) * nc + ob->cell];
                lam[(size_t)ob->fld * nc + ob->cell] +=
                    2.0 * d->lambda * wt * dz / (d->sig_o[ob->fld] * d->sig_o[ob->fld]);
            }
        if (d->ovl_levels && n > 0)
            for (int fl = 0; fl < NF; ++fl) {
                double ib = 1.0 / (d->sig_b[fl] * d->sig_b[fl]);
                for (int lj = 0; lj < s->ey; ++lj)
                    for (int li = 0; li < s->ex; ++li) {
                        int gi = imod(s->ei0 + li, nlon), gj = s->ej0 + lj;
                        long c = (long)lj * s->ex + li;
                        int m = d->nrowcov[gj] * d->ncolcov[gi] - 1;       /* other extended tiles holding the cell */
                        lam[(size_t)fl * nc + c] += 2.0 * d->mu * m * dtr[((size_t)n * NF + fl) * nc + c] * ib;
                    }
            }
        if (n > 0) {
            fill_padded(d, k, level - 1, traj + (size_t)(n - 1) * NF * nc, Zp, &r);
            region_forward(&d->m, &r, Zp, Za, Z1);
            interior_to_padded(s, &r, lam, L1);
            region_adjoint(&d->m, &r, Zp, Za, Z1, L1, A, HB, UB, L0);
            padded_to_interior(s, &r, L0, lam);
        }
    }
    for (int fl = 0; fl < NF; ++fl) {
        double ib = 1.0 / (d->sig_b[fl] * d->sig_b[fl]);
        for (int lj = 0; lj < s->ey; ++lj)
            for (int li = 0; li < s->ex; ++li) {
                int gi = imod(s->ei0 + li, nlon), gj = s->ej0 + lj;
                long c = (long)lj * s->ex + li;
                double dx = dtr[(size_t)fl * nc + c];
                double gsum = lam[(size_t)fl * nc + c];
                gsum += 2.0 * (s->jw == 0 ? 1.0 : d->bgw) * w_space(d, gi, gj) * dx * ib;       /* (25a) */
                for (int cb = 0; cb < d->nrowcov[gj]; ++cb)                                     /* (25c) case 1 */
                    for (int ca = 0; ca < d->ncolcov[gi]; ++ca) {
                        int a2 = d->colcov[4 * gi + ca], b2 = d->rowcov[4 * gj + cb];
                        if (a2 == s->a && b2 == s->b) continue;
                        gsum += 2.0 * d->mu * dx * ib;
                    }
                if (s->jw > 0) gsum += 2.0 * d->mu * dx * ib;                                   /* predecessor */
                out[(size_t)fl * nc + c] = d->sig_b[fl] * gsum;
            }
    }
    free(Zp); free(Za); free(Z1); free(dZp); free(dZa); free(dZ1); free(dtr);
    free(lam); free(L1); free(L0); free(A); free(HB); free(UB);
}

/* n_gn Gauss-Newton iterations on J_ji from w (updated in place); returns J_ji at the final w (one more
 * forward sweep, which also leaves the final trajectory in traj); *J0 = J_ji at the initial w. */
static double gn_run(const DD* d, int k, int n_gn, int n_cg, double* w, double* x, double* gx, double* traj,
                     double* J0)
{
    const Sub* s = &d->sub[k];
    const long n = NF * s->ncell;
    double* g = malloc(sizeof(double) * n); double* dw = malloc(sizeof(double) * n);
    double* rv = malloc(sizeof(double) * n); double* pv = malloc(sizeof(double) * n);
    double* Hp = malloc(sizeof(double) * n);
    CostParts cp;
    for (int it = 0; it < n_gn; ++it) {
        w_to_x(d, k, w, x);
        local_eval(d, k, x, &cp, gx, traj);
        if (it == 0 && J0) *J0 = cp.total;
        for (int fl = 0; fl < NF; ++fl)
            for (long q = 0; q < s->ncell; ++q) g[fl * s->ncell + q] = d->sig_b[fl] * gx[fl * s->ncell + q];
        for (long q = 0; q < n; ++q) { dw[q] = 0.0; rv[q] = -g[q]; pv[q] = rv[q]; }
        double rr = (double)ldot(rv, rv, n);
        for (int c = 0; c < n_cg && rr > 0.0; ++c) {
            local_gn_hessvec(d, k, traj, pv, Hp);
            double pHp = (double)ldot(pv, Hp, n);
            if (!(pHp > 0.0)) break;
            double al = rr / pHp;
            for (long q = 0; q < n; ++q) { dw[q] += al * pv[q]; rv[q] -= al * Hp[q]; }
            double rr2 = (double)ldot(rv, rv, n), be = rr2 / rr;
            for (long q = 0; q < n; ++q) pv[q] = rv[q] + be * pv[q];
            rr = rr2;
        }
        for (long q = 0; q < n; ++q) w[q] += dw[q];
    }
    w_to_x(d, k, w, x);
    local_eval(d, k, x, &cp, NULL, traj);
    if (n_gn == 0 && J0) *J0 = cp.total;
    free(g); free(dw); free(rv); free(pv); free(Hp);
    return cp.total;
}
/* Algorithm 1 with the Gauss-Newton local solver; same history layout as orc_run */
int orc_run_gn(void* h, int outer_iters, int n_gn, int n_cg, double* analysis, double* history)
{
    if (n_gn < 0 || n_cg < 0) return -1;
    return run_impl(h, outer_iters, analysis, history, 1, n_gn, n_cg);
}
/* test hook: H_GN p of subdomain k about the control x (p, out in w-space, [3][ncell]) */
int orc_gn_hessvec(void* h, int k, const double* x, const double* p, double* out)
{
    DD* d = h; if (!d->have_bg) return -3;
    if (k < 0 || k >= d->nsub) return -1;
    const Sub* s = &d->sub[k];
    CostParts cp;
    double* traj = malloc(sizeof(double) * NF * s->ncell * (s->e - s->s + 1));
    local_eval(d, k, x, &cp, NULL, traj);
    local_gn_hessvec(d, k, traj, p, out);
    free(traj);
    return 0;
}
/* test hook: n_gn Gauss-Newton iterations on subdomain k from the control x (in / out), n_cg CG iterations each */
int orc_gn_local(void* h, int k, int n_gn, int n_cg, double* x, double* J_first_last)
{
    DD* d = h; if (!d->have_bg) return -3;
    if (k < 0 || k >= d->nsub) return -1;
    const Sub* s = &d->sub[k]; const long n = NF * s->ncell;
    const double* ubs = ub_level(d, s->s);
    double* w = malloc(sizeof(double) * n); double* xx = malloc(sizeof(double) * n); double* gx = malloc(sizeof(double) * n);
    double* traj = malloc(sizeof(double) * n * (s->e - s->s + 1));
    for (int fl = 0; fl < NF; ++fl)
        for (int lj = 0; lj < s->ey; ++lj)
            for (int li = 0; li < s->ex; ++li) {
                int gi = imod(s->ei0 + li, d->m.nlon), gj = s->ej0 + lj;
                size_t c = (size_t)fl * s->ncell + (size_t)lj * s->ex + li;
                w[c] = (x[c] - ubs[gidx(d, fl, gj, gi)]) / d->sig_b[fl];
            }
    J_first_last[1] = gn_run(d, k, n_gn, n_cg, w, xx, gx, traj, &J_first_last[0]);
    memcpy(x, xx, sizeof(double) * n);
    free(w); free(xx); free(gx); free(traj);
    return 0;
}

/* ------------------------------------------------------------------ plain global 4D-Var ----
 * Written separately from the decomposition machinery (no Sub, no weights, no padded tiles):
 * minimise eq (6) in w = (x - x_b)/sigma_b with `rounds` restarts of n_inner L-BFGS iterations.
 * history[rounds+1] = J at the start and after each round. */
typedef struct { const DD* d; double* x; double* gx; } GlobCtx;
static void global_fn(void* ctx, const double* w, int want_grad, double* J, double* g)
{
    GlobCtx* c = ctx; const DD* d = c->d; size_t n1 = (size_t)d->m.nlon * d->m.nlat;
    for (int fl = 0; fl < NF; ++fl)
        for (size_t q = 0; q < n1; ++q) c->x[fl * n1 + q] = d->xb[fl * n1 + q] + d->sig_b[fl] * w[fl * n1 + q];
    *J = global_eval(d, c->x, want_grad ? c->gx : NULL, NULL);
    if (want_grad)
        for (int fl = 0; fl < NF; ++fl)
            for (size_t q = 0; q < n1; ++q) g[fl * n1 + q] = d->sig_b[fl] * c->gx[fl * n1 + q];
}
int orc_global_4dvar(void* h, int rounds, double* analysis, double* history)
{
    DD* d = h; if (!d->have_bg) return -3;
    size_t n1 = (size_t)d->m.nlon * d->m.nlat, n3 = NF * n1;
    double* w = calloc(n3, sizeof(double));
    GlobCtx c = { d, malloc(sizeof(double) * n3), malloc(sizeof(double) * n3) };
    history[0] = global_eval(d, d->xb, NULL, NULL);
    for (int l = 1; l <= rounds; ++l)
        history[l] = lbfgs_run((long)n3, d->lbfgs_m, d->n_inner, d->max_bt, d->c1, global_fn, &c, w, NULL);
    for (int fl = 0; fl < NF; ++fl)
        for (size_t q = 0; q < n1; ++q) analysis[fl * n1 + q] = d->xb[fl * n1 + q] + d->sig_b[fl] * w[fl * n1 + q];
    free(w); free(c.x); free(c.gx);
    return 0;
}
/* generic L-BFGS entry for the pin against a dense solve */
double orc_lbfgs(long n, int m, int n_iter, int max_bt, double c1, orc_evalfn fn, void* ctx, double* w)
{ return lbfgs_run(n, m, n_iter, max_bt, c1, fn, ctx, w, NULL); }

/* gradient-sweep timer for bench.py's cpu_baseline: evaluates J_ji and its gradient at the
 * current control for subs k0..k1-1 (OpenMP over subdomains) and returns processed
 * grid-point.steps (ext cells x window steps). */
double orc_sweep_range(void* h, int k0, int k1, double* cost_sum)
{
    DD* d = h; double pts = 0, cs = 0;
#pragma omp parallel for schedule(dynamic) reduction(+ : pts, cs)
    for (int k = k0; k < k1; ++k) {
        Sub* s = &d->sub[k]; long n = NF * s->ncell; double parts[6];
        double* x = malloc(sizeof(double) * n); double* g = malloc(sizeof(double) * n);
        orc_get_control(d, k, x);
        orc_eval_local_one(d, k, x, parts, g, NULL);
        pts += (double)s->ncell * (s->e - s->s); cs += parts[0];
        free(x); free(g);
    }
    *cost_sum = cs;
    return pts;
}
