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

struct CmSite { double Phi, rho_r, rhoe_r, rhoq_r, E_r, q_r, icvm_r; };
struct CmPrim { double rho, ir, u, v, w, q, K, p, pp, h, c2, drho; };

// geopotential + reference state at node n (k = its zeta index) of element e
template <int Nq, bool MOIST, int GEOM>
__device__ __forceinline__ void cm_load_site(const CmKP& p, int e, int n, int k, CmSite& s) {
  if constexpr (GEOM == 0) {
    const double2* t = reinterpret_cast<const double2*>(p.ztab + (size_t)(__ldg(p.erow + e) + k) * CM_ZTAB_W);
    double2 a = __ldg(t), b = __ldg(t + 1), c = __ldg(t + 2), d = __ldg(t + 3);
    s.Phi = a.x; s.rho_r = a.y; s.rhoe_r = b.x; s.rhoq_r = b.y; s.E_r = c.x; s.q_r = c.y; s.icvm_r = d.x;
  } else {
    const size_t idx = (size_t)e * CmNodes<Nq>::NP + n;
    s.Phi = p.th.grav * __ldg(p.geo + 10 * p.stride + idx);
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

// a1: primitive recovery (eq. 6-10, 13-14 with q_v = q_t) and p - p_r from state differences (R12)
template <bool MOIST>
__device__ __forceinline__ void cm_eos(const CmKP& p, const double* Y, const CmSite& s, CmPrim& P) {
  const CmThermo& th = p.th;
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

