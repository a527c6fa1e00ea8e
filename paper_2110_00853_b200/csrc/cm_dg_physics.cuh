// cm_dg_physics.cuh -- pointwise device functions shared by the hot kernels: geopotential / reference-state
// lookup, primitive recovery and EOS (a1), first- plus second-order fluxes (eq. 1-5, 16, 33-37).
#pragma once
#include "cm_dg_internal.h"

template <int Nq> struct CmNodes {
  static constexpr int NF = Nq * Nq;
  static constexpr int NP = Nq * Nq * Nq;
};

// 1/a and sqrt(a) to ~1 ulp from the MUFU seed plus two Newton steps: no slow-path branches (a > 0 here).
__device__ __forceinline__ double cm_rcp(double a) {
#ifdef CM_EXACT_MATH
  return 1.0 / a;
#endif
  double x;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(x) : "d"(a));
  double e = fma(-a, x, 1.0); x = fma(x, e, x);
  e = fma(-a, x, 1.0); x = fma(x, e, x);
  return x;
}
__device__ __forceinline__ double cm_sqrt(double a) {
  // the MUFU seed flushes subnormal inputs to zero (-> inf -> NaN after the Newton steps): squared strain rates of a
  // flow that has barely started (edge of the thermal bubble after one stage) do underflow that far, so arguments below
  // the fast path's safe range take the IEEE routine.  Rare, warp-uniform in practice.
  if (a < 1e-280) return (a > 0.0) ? sqrt(a) : 0.0;
#ifdef CM_EXACT_MATH
  return sqrt(a);
#endif
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
  double r = a * y, h = 0.5 * y;
  double e = fma(-r, h, 0.5); r = fma(r, e, r); h = fma(h, e, h);
  e = fma(-r, h, 0.5); r = fma(r, e, r);
  return (a > 0.0) ? r : 0.0;
}

struct CmSite { double Phi, rho_r, rhoe_r, rhoq_r, E_r, q_r, icvm_r, taus /* Rayleigh sponge coefficient (A5) */; };
struct CmPrim { double rho, ir, u, v, w, q, K, p, pp, h, c2, drho; };

// geopotential + reference state at node n (k = its zeta index) of element e
template <int Nq, bool MOIST, int GEOM>
__device__ __forceinline__ void cm_load_site(const CmKP& p, int e, int n, int k, CmSite& s) {
  if constexpr (GEOM == 0) {
    const double2* t = reinterpret_cast<const double2*>(p.ztab + (size_t)(__ldg(p.erow + e) + k) * CM_ZTAB_W);
    double2 a = __ldg(t), b = __ldg(t + 1), c = __ldg(t + 2), d = __ldg(t + 3);
    s.Phi = a.x; s.rho_r = a.y; s.rhoe_r = b.x; s.rhoq_r = b.y; s.E_r = c.x; s.q_r = c.y; s.icvm_r = d.x; s.taus = d.y;
  } else {
    const size_t idx = (size_t)e * CmNodes<Nq>::NP + n;
    s.Phi = p.th.grav * __ldg(p.geo + 10 * p.stride + idx);
    s.taus = __ldg(p.geo + 15 * p.stride + idx);
    if (p.use_ref) {
      s.rho_r = __ldg(p.ref + idx);
      s.rhoe_r = __ldg(p.ref + p.stride + idx);
      s.rhoq_r = MOIST ? __ldg(p.ref + 2 * p.stride + idx) : 0.0;
      s.q_r = MOIST ? s.rhoq_r * cm_rcp(s.rho_r) : 0.0;
      s.icvm_r = MOIST ? cm_rcp(p.th.c_vd + p.th.b * s.q_r) : p.th.icvd;
      s.E_r = s.rhoe_r - s.rho_r * s.Phi - s.rhoq_r * p.th.I_v0;
    } else {
      s.rho_r = s.rhoe_r = s.rhoq_r = s.E_r = s.q_r = 0.0; s.icvm_r = 0.0;
    }
  }
}

// Saturation adjustment (eq. 15): the root T of I*(T; rho, q_t) = I by Newton iterations with the analytical
// derivative, I* from eq. (7)-(8) with the excess q_t - q_v*(T, rho) as liquid, q_v* = p*(T) / (rho R_v T) and the
// closed-form p*(T) of a calorically perfect gas (Romps 2008).  Returns T; ql = liquid specific humidity.
__device__ __forceinline__ double cm_sat_q(const CmThermo& th, double T, double rho) {
  const double iT = 1.0 / T;
  return th.p_tr * pow(T * th.iT_tr, th.sx1) * exp(th.sx2 * (th.iT_tr - iT)) * iT / (rho * th.R_v);
}
// Safeguard: the root is bracketed from the start and the bracket shrinks with the sign of f at every iterate.
//   lo = unsaturated T: there the excess is still vapour, condensing it releases (c_vv - c_vl)(T - T_0) + I_v0 > 0 per
//        unit of water, so I*(lo) < I and f(lo) < 0;
//   hi = T with all of q_t liquid, T_0 + I / ((1 - q_t) c_vd + q_t c_vl): I*(T) - I_liquid(T) = q_v [(c_vv - c_vl)(T - T_0)
//        + I_v0] >= 0 for every T, so f(hi) >= 0.
// A Newton step that leaves [lo, hi] (or is not a number) is replaced by the midpoint, so a finite state always converges
// (bisection alone needs < 50 halvings of a bracket of tens of kelvin to reach 1e-14 T).  Iterates that stay inside, which
// is every step on the tested states, are the plain Newton iterates.  If the loop ends unconverged all the same (non-finite
// input), NaN is returned: it reaches the state and cm_dg_diagnostics counts it in n_nonfinite instead of a silently wrong
// pressure.
static __device__ __noinline__ double cm_sat_adjust(const CmThermo& th, double I, double rho, double qt, double& ql) {
  double T = th.T_0 + (I - qt * th.I_v0) / (th.c_vd + th.b * qt);
  if (qt <= cm_sat_q(th, T, rho)) { ql = 0.0; return T; }
  double lo = T, hi = th.T_0 + I / ((1.0 - qt) * th.c_vd + qt * th.c_vl);
  bool conv = false;
  for (int it = 0; it < 60; ++it) {
    const double qs = cm_sat_q(th, T, rho), dT0 = T - th.T_0;
    const double f = (1.0 - qt) * th.c_vd * dT0 + qs * (th.c_vv * dT0 + th.I_v0) + (qt - qs) * th.c_vl * dT0 - I;
    const double dqs = qs * ((th.Lv0 + th.dcp * dT0) / (th.R_v * T * T) - 1.0 / T);
    const double df = (1.0 - qt) * th.c_vd + qs * th.c_vv + (qt - qs) * th.c_vl + dqs * ((th.c_vv - th.c_vl) * dT0 + th.I_v0);
    if (f < 0.0) lo = fmax(lo, T); else hi = fmin(hi, T);
    double Tn = T - f / df;
    if (!(Tn >= lo && Tn <= hi)) Tn = 0.5 * (lo + hi);
    const double dT = T - Tn;
    T = Tn;
    if (fabs(dT) <= 1e-14 * T) { conv = true; break; }
  }
  if (!conv) T = __longlong_as_double(0x7ff8000000000000LL);
  ql = qt - cm_sat_q(th, T, rho);
  return T;
}
// pressure (eq. 13-14 with condensate), R_m and c_vm of moist air from (rho, I, q_t) under the saturation adjustment
__device__ __forceinline__ double cm_sat_pressure(const CmThermo& th, double rho, double I, double qt, double& Rm, double& cvm) {
  double ql;
  const double T = cm_sat_adjust(th, I, rho, qt, ql);
  Rm = th.R_d * (1.0 - qt) + th.R_v * (qt - ql);
  cvm = th.c_vd * (1.0 - qt) + th.c_vv * (qt - ql) + th.c_vl * ql;
  return rho * Rm * T;
}

// a1: primitive recovery (eq. 6-10, 13-14 with q_v = q_t) and p - p_r from state differences (R12)
// SAT: the kernel also carries the saturation-adjusted equation of state, chosen at run time by p.satadj
template <bool MOIST, bool SAT = false>
__device__ __forceinline__ void cm_eos(const CmKP& p, const double* Y, const CmSite& s, CmPrim& P) {
  const CmThermo& th = p.th;
  if constexpr (MOIST && SAT) {
    if (p.satadj) {
      P.rho = Y[0]; P.ir = 1.0 / Y[0];
      P.u = Y[1] * P.ir; P.v = Y[2] * P.ir; P.w = Y[3] * P.ir;
      P.q = Y[5] * P.ir;
      P.K = 0.5 * (Y[1] * P.u + Y[2] * P.v + Y[3] * P.w);
      const double I = Y[4] * P.ir - 0.5 * (P.u * P.u + P.v * P.v + P.w * P.w) - s.Phi;
      double Rm, cvm;
      P.p = cm_sat_pressure(th, Y[0], I, P.q, Rm, cvm);
      P.h = (Y[4] + P.p) * P.ir;
      P.c2 = (1.0 + Rm / cvm) * P.p * P.ir;
      if (p.use_ref) {
        // p_r = pressure of the resting reference state under the same equation of state (no R12 with condensate)
        double Rr, cr;
        P.pp = P.p - cm_sat_pressure(th, s.rho_r, s.rhoe_r / s.rho_r - s.Phi, s.rhoq_r / s.rho_r, Rr, cr);
        P.drho = Y[0] - s.rho_r;
      } else { P.pp = P.p; P.drho = Y[0]; }
      return;
    }
  }
  P.rho = Y[0];
  P.ir = cm_rcp(Y[0]);
  P.u = Y[1] * P.ir; P.v = Y[2] * P.ir; P.w = Y[3] * P.ir;
  const double rq = MOIST ? Y[5] : 0.0;
  P.q = MOIST ? rq * P.ir : 0.0;
  P.K = 0.5 * (Y[1] * P.u + Y[2] * P.v + Y[3] * P.w);
  double icvm, kappa;
  if (MOIST) { icvm = cm_rcp(th.c_vd + th.b * P.q); kappa = (th.R_d + th.a * P.q) * icvm; }
  else { icvm = th.icvd; kappa = th.kappa_d; }
  const double E = Y[4] - P.K - Y[0] * s.Phi - rq * th.I_v0;        // rho c_vm (T - T_0)
  P.p = kappa * E + th.T_0 * (th.R_d * Y[0] + th.a * rq);          // rho R_m T
  P.h = (Y[4] + P.p) * P.ir;
  P.c2 = (1.0 + kappa) * P.p * P.ir;
  if (p.use_ref) {
    const double drho = Y[0] - s.rho_r, drq = rq - s.rhoq_r;
    const double dE = (Y[4] - s.rhoe_r) - drho * s.Phi - drq * th.I_v0;
    const double dkappa = MOIST ? (P.q - s.q_r) * th.dk * icvm * s.icvm_r : 0.0;
    P.pp = kappa * dE - kappa * P.K + dkappa * s.E_r + th.T_0 * (th.R_d * drho + th.a * drq);
    P.drho = drho;
  } else {
    P.pp = P.p;
    P.drho = Y[0];
  }
}

// sum_c A_c (F1 + F2)[v][c] for all variables; g = packed SGS fluxes tau(xx,yy,zz,xy,xz,yz), J+D(3), d_q(3)
template <bool MOIST>
__device__ __forceinline__ void cm_flux_dir(const double* Y, const CmPrim& P, bool sgs, const double* g,
                                            double A0, double A1, double A2, double* Fn) {
  const double uA = A0 * P.u + A1 * P.v + A2 * P.w;
  double wA = uA, tA0 = 0.0, tA1 = 0.0, tA2 = 0.0, eA = 0.0, dqA = 0.0;
  if (sgs) {
    tA0 = g[0] * A0 + g[3] * A1 + g[4] * A2;
    tA1 = g[3] * A0 + g[1] * A1 + g[5] * A2;
    tA2 = g[4] * A0 + g[5] * A1 + g[2] * A2;
    eA = tA0 * P.u + tA1 * P.v + tA2 * P.w + (g[6] * A0 + g[7] * A1 + g[8] * A2);
    if (MOIST) { dqA = g[9] * A0 + g[10] * A1 + g[11] * A2; wA += dqA; }
  }
  Fn[0] = Y[0] * wA;
  Fn[1] = Y[1] * wA + P.pp * A0 + Y[0] * tA0;
  Fn[2] = Y[2] * wA + P.pp * A1 + Y[0] * tA1;
  Fn[3] = Y[3] * wA + P.pp * A2 + Y[0] * tA2;
  Fn[4] = (Y[4] + P.p) * uA + Y[0] * eA;
  if (MOIST) Fn[5] = Y[5] * uA + Y[0] * dqA;
}

// same for an axis-aligned direction A = s * e_AX (flat meshes)
template <bool MOIST, int AX>
__device__ __forceinline__ void cm_flux_axis(const double* Y, const CmPrim& P, bool sgs, const double* g,
                                             double s, double* Fn) {
  const double ud = (AX == 0) ? P.u : (AX == 1) ? P.v : P.w;
  double wA = ud, tA0 = 0.0, tA1 = 0.0, tA2 = 0.0, eA = 0.0, dqA = 0.0;
  if (sgs) {
    tA0 = (AX == 0) ? g[0] : (AX == 1) ? g[3] : g[4];
    tA1 = (AX == 0) ? g[3] : (AX == 1) ? g[1] : g[5];
    tA2 = (AX == 0) ? g[4] : (AX == 1) ? g[5] : g[2];
    eA = tA0 * P.u + tA1 * P.v + tA2 * P.w + g[6 + AX];
    if (MOIST) { dqA = g[9 + AX]; wA += dqA; }
  }
  Fn[0] = s * (Y[0] * wA);
  Fn[1] = s * (Y[1] * wA + ((AX == 0) ? P.pp : 0.0) + Y[0] * tA0);
  Fn[2] = s * (Y[2] * wA + ((AX == 1) ? P.pp : 0.0) + Y[0] * tA1);
  Fn[3] = s * (Y[3] * wA + ((AX == 2) ? P.pp : 0.0) + Y[0] * tA2);
  Fn[4] = s * ((Y[4] + P.p) * ud + Y[0] * eA);
  if (MOIST) Fn[5] = s * (Y[5] * ud + Y[0] * dqA);
}

// virtual potential temperature without condensate (eq. 40, reading R25) from pressure and 1 / rho
__device__ __forceinline__ double cm_theta_v(const CmThermo& th, double pr, double ir) {
  return pr * ir * th.iRd * pow(th.p_0 / pr, th.kap_pd);
}

// O5 / O11: eddy viscosity and packed SGS fluxes of one node.  Gr[s][c] = d s / d x_c for s = u, v, w, h_tot, q_t;
// thv, dthv_dz = theta_v and its vertical derivative (used when p.richardson); cs2d2 = (C_s Delta)^2 of eq. (38);
// d2 = squared mixing lengths of eq. (39c).  out = tau xx,yy,zz,xy,xz,yz | J + D x,y,z | d_q x,y,z  (eq. 34-37).
template <bool MOIST>
__device__ __forceinline__ void cm_closure(const CmKP& p, const double (&Gr)[5][3], double cs2d2, double d2x, double d2y,
                                           double d2z, double thv, double dthv_dz, double (&out)[12]) {
  const double Sxx = Gr[0][0], Syy = Gr[1][1], Szz = Gr[2][2];
  const double Sxy = 0.5 * (Gr[0][1] + Gr[1][0]), Sxz = 0.5 * (Gr[0][2] + Gr[2][0]), Syz = 0.5 * (Gr[1][2] + Gr[2][1]);
  const double ss2 = Sxx * Sxx + Syy * Syy + Szz * Szz + 2.0 * (Sxy * Sxy + Sxz * Sxz + Syz * Syz);   // S_ij S_ij
  double nu;
  if (p.sgs == 2) {
    // Vreman (eq. 39a-d): beta_ij = Delta_m^2 u_i,m u_j,m; B = second invariant of beta
    double b[3][3];
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int j = i; j < 3; ++j) b[i][j] = d2x * Gr[i][0] * Gr[j][0] + d2y * Gr[i][1] * Gr[j][1] + d2z * Gr[i][2] * Gr[j][2];
    const double B = b[0][0] * b[1][1] + b[0][0] * b[2][2] + b[1][1] * b[2][2] - (b[0][2] * b[0][2] + b[0][1] * b[0][1] + b[1][2] * b[1][2]);
    double aa = 0.0;
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int j = 0; j < 3; ++j) aa += Gr[i][j] * Gr[i][j];
    nu = (aa > 0.0 && B > 0.0) ? 2.5 * p.cs2 * sqrt(B / aa) : 0.0;
  } else {
    nu = cs2d2 * cm_sqrt(2.0 * ss2);                                       // eq. (38)
  }
  if (p.richardson) {
    // eq. (40): Ri = (g / theta_v) (d theta_v / dz) / |S|^2, |S|^2 = 2 S_ij S_ij; f_b = max(0, 1 - Ri / Pr_t)^(1/4)
    const double N2 = (p.th.grav / thv) * dthv_dz;
    double fb = 1.0;
    if (N2 > 0.0) {
      const double t = 1.0 - (N2 / (2.0 * ss2)) * p.inv_Pr;
      fb = (t > 0.0) ? sqrt(sqrt(t)) : 0.0;
    }
    nu *= fb;
  }
  const double m2nu = -2.0 * nu, mDt = -nu * p.inv_Pr;
  out[0] = m2nu * Sxx; out[1] = m2nu * Syy; out[2] = m2nu * Szz; out[3] = m2nu * Sxy; out[4] = m2nu * Sxz; out[5] = m2nu * Syz;
  out[6] = mDt * Gr[3][0]; out[7] = mDt * Gr[3][1]; out[8] = mDt * Gr[3][2];
  out[9] = MOIST ? mDt * Gr[4][0] : 0.0; out[10] = MOIST ? mDt * Gr[4][1] : 0.0; out[11] = MOIST ? mDt * Gr[4][2] : 0.0;
}

// A . F1(Y) for all variables (first-order flux only; A = sJ n)
template <bool MOIST>
__device__ __forceinline__ void cm_flux1_dir(const double* Y, const CmPrim& P, double A0, double A1, double A2, double* Fn) {
  const double uA = A0 * P.u + A1 * P.v + A2 * P.w;
  Fn[0] = Y[0] * uA;
  Fn[1] = Y[1] * uA + P.pp * A0; Fn[2] = Y[2] * uA + P.pp * A1; Fn[3] = Y[3] * uA + P.pp * A2;
  Fn[4] = (Y[4] + P.p) * uA;
  if (MOIST) Fn[5] = Y[5] * uA;
}

// HLLC flux (Toro, Spruce & Speares 1994): Fs = sJ n.F1* from the two states, A = sJ n, AFm / AFp = A.F1 of the
// two sides.  Wave speeds S_L = min(u_L - c_L, u_R - c_R), S_R = max(u_L + c_L, u_R + c_R); p' in the momentum
// flux, full p in the energy relation (reading R27 of DESIGN.md).
template <bool MOIST>
__device__ __forceinline__ void cm_hllc(const double* Ym, const CmPrim& Pm, const double* AFm, const double* Yp, const CmPrim& Pp,
                                        const double* AFp, const double* A, double sJ, double* Fs) {
  constexpr int NV = MOIST ? 6 : 5;
  const double isJ = 1.0 / sJ;
  const double n0 = A[0] * isJ, n1 = A[1] * isJ, n2 = A[2] * isJ;
  const double unm = Pm.u * n0 + Pm.v * n1 + Pm.w * n2, unp = Pp.u * n0 + Pp.v * n1 + Pp.w * n2;
  const double cm_ = sqrt(Pm.c2), cp = sqrt(Pp.c2);
  const double SL = fmin(unm - cm_, unp - cp), SR = fmax(unm + cm_, unp + cp);
  if (SL >= 0.0) { for (int v = 0; v < NV; ++v) Fs[v] = AFm[v]; return; }
  if (SR <= 0.0) { for (int v = 0; v < NV; ++v) Fs[v] = AFp[v]; return; }
  const double Sstar = ((Pp.pp - Pm.pp) + Ym[0] * unm * (SL - unm) - Yp[0] * unp * (SR - unp)) /
                       (Ym[0] * (SL - unm) - Yp[0] * (SR - unp));
  const bool left = Sstar >= 0.0;
  const double* Y = left ? Ym : Yp; const CmPrim& P = left ? Pm : Pp;
  const double un = left ? unm : unp, SK = left ? SL : SR;
  const double* AF = left ? AFm : AFp;
  // the jump U*_K - U_K formed analytically (rho* - rho = rho (S* - u_n) / (S_K - S*)): no cancellation of O(rho c) terms
  const double ds = Sstar - un;
  const double rs = Y[0] * (SK - un) / (SK - Sstar), drho = Y[0] * ds / (SK - Sstar);
  double dU[6];
  dU[0] = drho;
  dU[1] = drho * P.u + rs * ds * n0; dU[2] = drho * P.v + rs * ds * n1; dU[3] = drho * P.w + rs * ds * n2;
  dU[4] = drho * (Y[4] / Y[0]) + rs * ds * (Sstar + P.p / (Y[0] * (SK - un)));
  if (MOIST) dU[5] = drho * P.q;
  for (int v = 0; v < NV; ++v) Fs[v] = AF[v] + sJ * (SK * dU[v]);
}

// Surface fluxes of the bottom wall (face 4), added to the wall's lifted flux term r = -sJ n.F* (+ own side):
//   energy  n_in . rho (J + D) = SHF + LHF (p.shf holds the sum), water and with it mass E = n_in . (rho d_qv)
//   (P:L672-679), momentum  n_in . (rho tau) = -rho C_d |u_p,int| u_p,int  (eq. A2) with u_p,int the
//   wall-parallel velocity at the first layer of interior nodes: Yi = state of the node above the wall node (stride si).
// A = outward sJ n of the wall node, rho = density at the wall node.
template <bool MOIST>
__device__ __forceinline__ void cm_surface_flux(const CmKP& p, const double* A, double sJ, double rho, const double* Yi, int si,
                                                double* r) {
  r[4] += sJ * p.shf;
  if (MOIST) { r[0] += sJ * p.evap; r[5] += sJ * p.evap; }
  if (p.drag_cd > 0.0) {
    const double ir = cm_rcp(Yi[0]), isJ = cm_rcp(sJ);
    const double u = Yi[si] * ir, v = Yi[2 * si] * ir, w = Yi[3 * si] * ir;
    const double n0 = A[0] * isJ, n1 = A[1] * isJ, n2 = A[2] * isJ;
    const double un = u * n0 + v * n1 + w * n2;
    const double u0 = u - un * n0, u1 = v - un * n1, u2 = w - un * n2;
    const double c = sJ * rho * p.drag_cd * cm_sqrt(u0 * u0 + u1 * u1 + u2 * u2);
    r[1] -= c * u0; r[2] -= c * u1; r[3] -= c * u2;
  }
}

// Roe flux (Roe 1981): Fs = sJ n.F1* = (1/2)(A.F1^- + A.F1^+) - (1/2) sJ sum_k |lambda_k| alpha_k r_k with the
// sqrt(rho)-weighted averages of u, h_tot and q.  With the mixture frozen at q~ the EOS is an ideal gas with
// gamma - 1 = kappa~ and the energy shifted by s~ = Phi + q~ I_v0 - c_vm T_0, so c~^2 = kappa~ (H~ - s~ - |u~|^2 / 2);
// rho q is a passive wave of speed u~_n.  Phi = geopotential of the face node.
template <bool MOIST>
__device__ __forceinline__ void cm_roe(const CmKP& p, const double* Ym, const CmPrim& Pm, const double* AFm, const double* Yp,
                                       const CmPrim& Pp, const double* AFp, const double* A, double sJ, double Phi, double* Fs) {
  constexpr int NV = MOIST ? 6 : 5;
  const CmThermo& th = p.th;
  const double isJ = 1.0 / sJ;
  const double n[3] = {A[0] * isJ, A[1] * isJ, A[2] * isJ};
  const double wm = sqrt(Ym[0]), wp = sqrt(Yp[0]), iw = 1.0 / (wm + wp);
  const double um[3] = {Pm.u, Pm.v, Pm.w}, up[3] = {Pp.u, Pp.v, Pp.w};
  double ut[3], du[3], un = 0.0, K = 0.0, dun = 0.0;
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    ut[i] = (wm * um[i] + wp * up[i]) * iw; du[i] = up[i] - um[i];
    un += ut[i] * n[i]; K += 0.5 * ut[i] * ut[i]; dun += du[i] * n[i];
  }
  const double H = (wm * Pm.h + wp * Pp.h) * iw;
  const double q = MOIST ? (wm * Pm.q + wp * Pp.q) * iw : 0.0;
  const double cvm = th.c_vd + th.b * q, kappa = (th.R_d + th.a * q) / cvm;
  const double sh = Phi + q * th.I_v0 - cvm * th.T_0;
  const double c2 = kappa * (H - sh - K), cs = sqrt(c2);
  const double rt = wm * wp;
  const double drho = Yp[0] - Ym[0], dp = Pp.pp - Pm.pp;
  const double a1 = (dp - rt * cs * dun) / (2.0 * c2), a5 = (dp + rt * cs * dun) / (2.0 * c2), a2 = drho - dp / c2;
  const double l1 = fabs(un - cs), l2 = fabs(un), l5 = fabs(un + cs);
  double D[6];
  D[0] = l1 * a1 + l2 * a2 + l5 * a5;
  double udu = 0.0;
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    const double shr = du[i] - dun * n[i];
    D[1 + i] = l1 * a1 * (ut[i] - cs * n[i]) + l2 * (a2 * ut[i] + rt * shr) + l5 * a5 * (ut[i] + cs * n[i]);
    udu += ut[i] * shr;
  }
  D[4] = l1 * a1 * (H - cs * un) + l2 * (a2 * (K + sh) + rt * udu) + l5 * a5 * (H + cs * un);
  if (MOIST) D[5] = (l1 * a1 + l2 * a2 + l5 * a5) * q + l2 * rt * (Pp.q - Pm.q);
#pragma unroll
  for (int v = 0; v < NV; ++v) Fs[v] = 0.5 * (AFm[v] + AFp[v]) - 0.5 * sJ * D[v];
}

template <int NV>
__device__ __forceinline__ void cm_load_state(const double* __restrict__ Q, long long stride, size_t idx, double* Y) {
#pragma unroll
  for (int v = 0; v < NV; ++v) Y[v] = __ldg(Q + v * stride + idx);
}

// face geometry helper: A = sgn * Ja^d at own face node (outward, unnormalised: sJ * n)
template <int Nq, int GEOM>
__device__ __forceinline__ void cm_face_vector(const CmKP& p, int e, int n, int d, double sgn, double* A) {
  if constexpr (GEOM == 0) {
    A[0] = (d == 0) ? sgn * p.cA[0] : 0.0; A[1] = (d == 1) ? sgn * p.cA[1] : 0.0; A[2] = (d == 2) ? sgn * p.cA[2] : 0.0;
  } else {
    const size_t idx = (size_t)e * CmNodes<Nq>::NP + n;
#pragma unroll
    for (int c = 0; c < 3; ++c) A[c] = sgn * __ldg(p.geo + (size_t)(3 * d + c) * p.stride + idx);
  }
}

