// model_math.cuh -- per-cell arithmetic of one model step Phi and of its adjoint (gather form).
//
// Phi is the operator-split one-step scheme of DESIGN.md R3 on the Turkel-Zwas member p=q=1,
// alpha=0 of PAPER.md l.971-989, for the shallow-water equations on the sphere eq (60)-(62)
// l.945-954 in advective form:
//   stage A : x^a = x - dt [cz u (x_E - x_W) + cm v (x_N - x_S)] + kappa L(x),  x in {h,u,v}
//   stage B : h^1 = h^a - dt h^a [cz (u^a_E - u^a_W) + cm (r+ v^a_N - r- v^a_S)]
//             u^1 = u^a + dt [-g cz (h^1_E - h^1_W) + (f + t u^a) v^a]
//             v^1 = v^a + dt [-g cm (h^1_N - h^1_S) - (f + t u^1) u^1]
// with dt folded into the row tables.  The adjoint (eq (3)-(4) l.91-98) is written so that every
// thread GATHERS the value of its own cell (no scatter, no atomics):
//   UB  = ub1 - (dtf + 2 dtt u^1) vb1
//   HB  = hb1 + gdtcm (vb1_N - vb1_S) + gdtcz (UB_E - UB_W)
//   P   = -h^a HB
//   A_h = HB (1 - Ddt),  Ddt = dtcz (u^a_E - u^a_W) + dtcm (r+ v^a_N - r- v^a_S)
//   A_u = UB (1 + dtt v^a) + dtcz (P_W - P_E)
//   A_v = vb1 + UB (dtf + dtt u^a) + dtcm (r+_{j-1} P_S - r-_{j+1} P_N)
//   L0_x = A_x (1 - 4 kappa) + A_x,W (kappa - dtcz u_W) + A_x,E (kappa + dtcz u_E)
//                            + A_x,S (kappa - dtcm v_S) + A_x,N (kappa + dtcm v_N)
//   L0_u -= dtcz sum_x (x_E - x_W) A_x ;   L0_v -= dtcm sum_x (x_N - x_S) A_x
// A reflective pole wall (R4) enters as a mirrored neighbour row with v, vb1, A_v
// negated; the callers pass those mirrored values.
#pragma once

__device__ __forceinline__ double mm_stageA(double x, double xE, double xW, double xN, double xS,
                                            double cu /* dtcz*u0 */, double cv /* dtcm*v0 */,
                                            double kap)
{
    return x - (cu * (xE - xW) + cv * (xN - xS)) + kap * (xE + xW + xN + xS - 4.0 * x);
}
// Ddt: the divergence bracket times dt (vaN, vaS already carry the wall sign)
__device__ __forceinline__ double mm_div(double uaE, double uaW, double vaN, double vaS,
                                         double dtcz, double dtcm, double rp, double rm)
{
    return dtcz * (uaE - uaW) + dtcm * (rp * vaN - rm * vaS);
}
__device__ __forceinline__ double mm_h1(double ha, double Ddt) { return ha - ha * Ddt; }
__device__ __forceinline__ double mm_u1(double ua, double va, double h1E, double h1W,
                                        double gdtcz, double dtf, double dtt)
{
    return ua - gdtcz * (h1E - h1W) + (dtf + dtt * ua) * va;
}
__device__ __forceinline__ double mm_v1(double va, double u1, double h1N, double h1S,
                                        double gdtcm, double dtf, double dtt)
{
    return va - gdtcm * (h1N - h1S) - (dtf + dtt * u1) * u1;
}

// ---- adjoint, gather form
__device__ __forceinline__ double mm_UB(double ub1, double vb1, double u1, double dtf, double dtt)
{
    return ub1 - (dtf + 2.0 * dtt * u1) * vb1;
}
__device__ __forceinline__ double mm_HB(double hb1, double vbN, double vbS, double UBE, double UBW,
                                        double gdtcm, double gdtcz)
{
    return hb1 + gdtcm * (vbN - vbS) + gdtcz * (UBE - UBW);
}
__device__ __forceinline__ double mm_Ah(double HB, double Ddt) { return HB * (1.0 - Ddt); }
__device__ __forceinline__ double mm_Au(double UB, double va, double PW, double PE, double dtt,
                                        double dtcz)
{
    return UB * (1.0 + dtt * va) + dtcz * (PW - PE);
}
// PSr = r+_{j-1} P_S (or r-_j P_c at the south wall), PNr = r-_{j+1} P_N (or r+_j P_c at the north wall)
__device__ __forceinline__ double mm_Av(double vb1, double UB, double ua, double PSr, double PNr,
                                        double dtf, double dtt, double dtcm)
{
    return vb1 + UB * (dtf + dtt * ua) + dtcm * (PSr - PNr);
}
// transport part of L0 for one field: the 5-point transposed advection-diffusion stencil
__device__ __forceinline__ double mm_L0(double Ac, double AW, double AE, double AS, double AN,
                                        double cuW /* dtcz*u0_W */, double cuE, double cvS
                                        /* dtcm*v0_S */, double cvN, double kap)
{
    return Ac * (1.0 - 4.0 * kap) + AW * (kap - cuW) + AE * (kap + cuE) + AS * (kap - cvS) +
           AN * (kap + cvN);
}
