// cm_dg_kernels.cuh -- the two hot kernels of the DG right-hand side (sm_100a, fp64 CUDA cores).
//
//   cm_gradient_kernel : a1 + a2 of the scope table -- primitive recovery, BR1 auxiliary gradient with
//                        central flux (eq. 28-31; walls A6-A8) and the
//                        Smagorinsky-Lilly closure (eq. 33-38).  Output: the SGS fluxes per unit
//                        mass tau (6), J+D (3), d_q (3) -- or the 15 raw gradients (diagnostic mode).
//   cm_tendency_kernel : a1 + a3 + a4 + a5 -- fluxes F1 + F2 (eq. 1-5, 16), strong-form volume term
//                        (eq. 32), Rusanov / central face fluxes with lift (eq. 27), gravity
//                        source (eq. 4) and the fused 2N-storage LSRK update.
//
// Work decomposition (both kernels): one CTA owns EPB consecutive elements; one thread owns the column
// (i, j, 0..N) of one element.  The zeta-direction contraction runs in registers with D as constant-bank
// operands; xi/eta contractions read an element tile staged in shared memory; every thread evaluates
// exactly 6 face nodes (its own two zeta-face nodes and one node of each lateral face), so the face
// work is balanced across lanes.  Neighbour traces come straight from global memory (L2).
#pragma once
#include "cm_dg_internal.h"
#include "cm_dg_physics.cuh"

template <int Nq> struct CmCfg {
  static constexpr int NF = Nq * Nq;
  static constexpr int NP = Nq * Nq * Nq;
  static constexpr int EPB = (Nq == 3) ? 14 : (Nq == 4) ? 8 : (Nq == 5) ? 5 : (Nq == 6) ? 3 : 2;
  static constexpr int THREADS = EPB * NF;
};

// ------------------------------------------------------------------------------------------------
// a2: auxiliary gradient.  delta[v] = s*[v] - s^-[v] at one face node (central flux or wall rule)
// ------------------------------------------------------------------------------------------------
template <int Nq, bool MOIST, int GEOM>
__device__ __forceinline__ void cm_grad_face_delta(const CmKP& p, int e, int nb, int nm, int np_, int kp,
                                                   int d, double sgn, const double* sm, double* delta) {
  constexpr int NV = MOIST ? 6 : 5;
  if (nb >= 0) {
    double Y[6]; CmSite st; CmPrim P;
    cm_load_state<NV>(p.Q, p.stride, (size_t)nb * CmCfg<Nq>::NP + np_, Y);
    cm_load_site<Nq, MOIST, GEOM>(p, nb, np_, kp, st);
    cm_eos<MOIST>(p, Y, st, P);
    delta[0] = 0.5 * (P.u - sm[0]); delta[1] = 0.5 * (P.v - sm[1]); delta[2] = 0.5 * (P.w - sm[2]);
    delta[3] = 0.5 * (P.h - sm[3]); delta[4] = MOIST ? 0.5 * (P.q - sm[4]) : 0.0;
  } else {
    // wall: u_bc = u^- - (n.u^-) n  (A6); scalars unchanged (A8)
    double A[3]; cm_face_vector<Nq, GEOM>(p, e, nm, d, sgn, A);
    const double ua = (sm[0] * A[0] + sm[1] * A[1] + sm[2] * A[2]) / (A[0] * A[0] + A[1] * A[1] + A[2] * A[2]);
    delta[0] = -ua * A[0]; delta[1] = -ua * A[1]; delta[2] = -ua * A[2]; delta[3] = 0.0; delta[4] = 0.0;
  }
}

template <int Nq, bool MOIST, int GEOM>
__global__ void __launch_bounds__(CmCfg<Nq>::THREADS) cm_gradient_kernel(const __grid_constant__ CmKP p) {
  using C = CmCfg<Nq>;
  constexpr int NF = C::NF, NP = C::NP, N = Nq - 1;
  constexpr int NV = MOIST ? 6 : 5;
  constexpr int NS = MOIST ? 5 : 4;          // gradient variables u, v, w, h_tot, [q_t]
  extern __shared__ double smem[];
  double* Dsh = smem;                                      // [Nq][Nq]
  double* s_sh = Dsh + Nq * Nq;                            // [EPB][NS][NP]
  double* fbuf = s_sh + C::EPB * NS * NP;                  // [EPB][4][NF][NS]

  const int tid = threadIdx.x;
  const int el = tid / NF, t2 = tid % NF, i = t2 % Nq, j = t2 / Nq;
  const int e = blockIdx.x * C::EPB + el;
  const bool active = e < p.Ne;
  if (tid < Nq * Nq) Dsh[tid] = p.D[tid / Nq][tid % Nq];

  double* ssh = s_sh + el * NS * NP;
  double* fb = fbuf + el * 4 * NF * NS;
  double sv[Nq][NS];
  if (active) {
#pragma unroll
    for (int k = 0; k < Nq; ++k) {
      const int n = t2 + NF * k;
      double Y[6]; CmSite st; CmPrim P;
      cm_load_state<NV>(p.Q, p.stride, (size_t)e * NP + n, Y);
      cm_load_site<Nq, MOIST, GEOM>(p, e, n, k, st);
      cm_eos<MOIST>(p, Y, st, P);
      sv[k][0] = P.u; sv[k][1] = P.v; sv[k][2] = P.w; sv[k][3] = P.h;
      if (MOIST) sv[k][NS - 1] = P.q;
#pragma unroll
      for (int v = 0; v < NS; ++v) ssh[v * NP + n] = sv[k][v];
    }
  }
  __syncthreads();
  double Di[Nq], Dj[Nq];
#pragma unroll
  for (int m = 0; m < Nq; ++m) { Di[m] = Dsh[i * Nq + m]; Dj[m] = Dsh[j * Nq + m]; }

  double dz0[NS], dzN[NS];
  if (active) {
    const int* nbr = p.nbr + (size_t)e * 6;
    // lateral faces: this thread takes node (a, b) = (i, j) of faces 0..3
#pragma unroll
    for (int f = 0; f < 4; ++f) {
      const int d = f >> 1;
      const int at = (f & 1) ? N : 0, ot = N - at;
      const int nm = (d == 0) ? (at + Nq * i + NF * j) : (i + Nq * at + NF * j);
      const int np_ = (d == 0) ? (ot + Nq * i + NF * j) : (i + Nq * ot + NF * j);
      double sm[5], delta[5];
#pragma unroll
      for (int v = 0; v < NS; ++v) sm[v] = ssh[v * NP + nm];
      if (!MOIST) sm[4] = 0.0;
      cm_grad_face_delta<Nq, MOIST, GEOM>(p, e, __ldg(nbr + f), nm, np_, j, d, (f & 1) ? 1.0 : -1.0, sm, delta);
#pragma unroll
      for (int v = 0; v < NS; ++v) fb[(f * NF + t2) * NS + v] = delta[v];
    }
    // zeta faces: own column ends
    {
      double sm[5], delta[5];
#pragma unroll
      for (int v = 0; v < NS; ++v) sm[v] = sv[0][v];
      if (!MOIST) sm[4] = 0.0;
      cm_grad_face_delta<Nq, MOIST, GEOM>(p, e, __ldg(nbr + 4), t2, t2 + NF * N, N, 2, -1.0, sm, delta);
#pragma unroll
      for (int v = 0; v < NS; ++v) dz0[v] = delta[v];
#pragma unroll
      for (int v = 0; v < NS; ++v) sm[v] = sv[N][v];
      cm_grad_face_delta<Nq, MOIST, GEOM>(p, e, __ldg(nbr + 5), t2 + NF * N, t2, 0, 2, 1.0, sm, delta);
#pragma unroll
      for (int v = 0; v < NS; ++v) dzN[v] = delta[v];
    }
  }
  __syncthreads();
  if (!active) return;

#pragma unroll
  for (int k = 0; k < Nq; ++k) {
    const int n = t2 + NF * k;
    const size_t idx = (size_t)e * NP + n;
    // metric terms a^d_c = Ja^d_c / J and lift vectors
    double Ja[3][3], invJ, cs2d2;
    if constexpr (GEOM == 0) {
      invJ = p.invJ; cs2d2 = p.cs2delta2;
    } else {
#pragma unroll
      for (int d = 0; d < 3; ++d)
#pragma unroll
        for (int c = 0; c < 3; ++c) Ja[d][c] = __ldg(p.geo + (size_t)(3 * d + c) * p.stride + idx);
      invJ = __ldg(p.geo + 9 * p.stride + idx);
      cs2d2 = __ldg(p.geo + 11 * p.stride + idx);
    }
    double G[5][3];
#pragma unroll
    for (int v = 0; v < NS; ++v) {
      double dr = 0.0, ds = 0.0, dt = 0.0;
#pragma unroll
      for (int m = 0; m < Nq; ++m) {
        dr += Di[m] * ssh[v * NP + m + Nq * j + NF * k];
        ds += Dj[m] * ssh[v * NP + i + Nq * m + NF * k];
        dt += p.D[k][m] * sv[m][v];
      }
      // surface lift: (1 / (w_0 J)) * (sgn Ja^d) * delta, faces in the fixed order xi-, xi+, eta-, eta+, zeta-, zeta+
      const double w0i = p.inv_w0;
      if (i == 0) dr -= w0i * fb[(0 * NF + j + Nq * k) * NS + v];
      if (i == N) dr += w0i * fb[(1 * NF + j + Nq * k) * NS + v];
      if (j == 0) ds -= w0i * fb[(2 * NF + i + Nq * k) * NS + v];
      if (j == N) ds += w0i * fb[(3 * NF + i + Nq * k) * NS + v];
      if (k == 0) dt -= w0i * dz0[v];
      if (k == N) dt += w0i * dzN[v];
      if constexpr (GEOM == 0) {
        G[v][0] = (p.cA[0] * invJ) * dr; G[v][1] = (p.cA[1] * invJ) * ds; G[v][2] = (p.cA[2] * invJ) * dt;
      } else {
#pragma unroll
        for (int c = 0; c < 3; ++c) G[v][c] = invJ * (Ja[0][c] * dr + Ja[1][c] * ds + Ja[2][c] * dt);
      }
    }
    if (!MOIST) { G[4][0] = G[4][1] = G[4][2] = 0.0; }
    if (p.mode == 1) {
#pragma unroll
      for (int v = 0; v < 5; ++v)
#pragma unroll
        for (int c = 0; c < 3; ++c) p.Gout[(size_t)(3 * v + c) * p.stride + idx] = G[v][c];
    } else {
      // eq. (33)-(38): S, nu_t = (C_s Delta)^2 sqrt(2 S:S), D_t = nu_t / Pr_t; store tau, J + D, d_q
      const double Sxx = G[0][0], Syy = G[1][1], Szz = G[2][2];
      const double Sxy = 0.5 * (G[0][1] + G[1][0]), Sxz = 0.5 * (G[0][2] + G[2][0]), Syz = 0.5 * (G[1][2] + G[2][1]);
      const double ss = Sxx * Sxx + Syy * Syy + Szz * Szz + 2.0 * (Sxy * Sxy + Sxz * Sxz + Syz * Syz);
      const double nu = cs2d2 * cm_sqrt(2.0 * ss);
      const double m2nu = -2.0 * nu, mDt = -nu * p.inv_Pr;
      double* o = p.Gout + idx;
      o[0] = m2nu * Sxx; o[p.stride] = m2nu * Syy; o[2 * p.stride] = m2nu * Szz;
      o[3 * p.stride] = m2nu * Sxy; o[4 * p.stride] = m2nu * Sxz; o[5 * p.stride] = m2nu * Syz;
      o[6 * p.stride] = mDt * G[3][0]; o[7 * p.stride] = mDt * G[3][1]; o[8 * p.stride] = mDt * G[3][2];
      if (MOIST) { o[9 * p.stride] = mDt * G[4][0]; o[10 * p.stride] = mDt * G[4][1]; o[11 * p.stride] = mDt * G[4][2]; }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// a3-a5: tendency.  One face node: r[v] = sgn*Ft^- [v] - sJ F*[v]   (so that dQ += r / (w_0 J))
// ------------------------------------------------------------------------------------------------
template <int Nq, bool MOIST, int GEOM>
__device__ __forceinline__ void cm_tend_face(const CmKP& p, int e, int nb, int f, int nm, int np_, int kp,
                                             const double* Ym, const double* Ftm /* sgn * Ft^d at the node */,
                                             double c2m, double* r) {
  constexpr int NV = MOIST ? 6 : 5;
  constexpr int NG = MOIST ? 12 : 9;
  constexpr int NP = CmCfg<Nq>::NP;
  const int d = f >> 1;
  const double sgn = (f & 1) ? 1.0 : -1.0;
  double A[3]; cm_face_vector<Nq, GEOM>(p, e, nm, d, sgn, A);
  const double sJ = (GEOM == 0) ? p.cA[d] : sqrt(A[0] * A[0] + A[1] * A[1] + A[2] * A[2]);
  const double irm = cm_rcp(Ym[0]);
  const double uAm = (Ym[1] * A[0] + Ym[2] * A[1] + Ym[3] * A[2]) * irm;     // sJ * (u^- . n)
  const double cm_ = cm_sqrt(c2m);
  if (nb >= 0) {
    double Yp[6], g[12]; CmSite st; CmPrim P;
    const size_t idp = (size_t)nb * NP + np_;
    cm_load_state<NV>(p.Q, p.stride, idp, Yp);
    if (p.sgs) cm_load_state<NG>(p.G, p.stride, idp, g);
    cm_load_site<Nq, MOIST, GEOM>(p, nb, np_, kp, st);
    cm_eos<MOIST>(p, Yp, st, P);
    double Fp[6];
    if constexpr (GEOM == 0) {
      if (d == 0) cm_flux_axis<MOIST, 0>(Yp, P, p.sgs, g, A[0], Fp);
      else if (d == 1) cm_flux_axis<MOIST, 1>(Yp, P, p.sgs, g, A[1], Fp);
      else cm_flux_axis<MOIST, 2>(Yp, P, p.sgs, g, A[2], Fp);
    } else {
      cm_flux_dir<MOIST>(Yp, P, p.sgs, g, A[0], A[1], A[2], Fp);
    }
    const double uAp = A[0] * P.u + A[1] * P.v + A[2] * P.w;
    const double lamsJ = fmax(fabs(uAm) + cm_ * sJ, fabs(uAp) + cm_sqrt(P.c2) * sJ);   // sJ * lambda (R2)
#pragma unroll
    for (int v = 0; v < NV; ++v) r[v] = 0.5 * (Ftm[v] - Fp[v]) - 0.5 * lamsJ * (Ym[v] - Yp[v]);
  } else {
    // free-slip wall (A6-A7): Rusanov flux against the mirrored state is [0; (p' + rho u_n (u_n + lambda)) n; 0; 0],
    // all second-order normal fluxes vanish (R10) except the prescribed bottom energy flux.
    CmSite st; CmPrim P;
    cm_load_site<Nq, MOIST, GEOM>(p, e, nm, (f < 4) ? kp : ((f == 4) ? 0 : Nq - 1), st);
    cm_eos<MOIST>(p, Ym, st, P);
    const double isJ = 1.0 / sJ;
    const double un = uAm * isJ;
    const double lam = fabs(un) + cm_;
    const double mom = (P.pp + Ym[0] * un * (un + lam));
#pragma unroll
    for (int v = 0; v < NV; ++v) r[v] = Ftm[v];
    r[1] -= mom * A[0]; r[2] -= mom * A[1]; r[3] -= mom * A[2];
    if (f == 4) r[4] += sJ * p.shf;
  }
}

template <int Nq, bool MOIST, int GEOM>
__global__ void __launch_bounds__(CmCfg<Nq>::THREADS) cm_tendency_kernel(const __grid_constant__ CmKP p) {
  using C = CmCfg<Nq>;
  constexpr int NF = C::NF, NP = C::NP, N = Nq - 1;
  constexpr int NV = MOIST ? 6 : 5;
  constexpr int NG = MOIST ? 12 : 9;
  extern __shared__ double smem[];
  double* Dsh = smem;                                 // [Nq][Nq]
  double* F1sh = Dsh + Nq * Nq;                       // [EPB][NV][NP]  contravariant flux, xi direction
  double* F2sh = F1sh + C::EPB * NV * NP;             // [EPB][NV][NP]  eta direction
  double* c2sh = F2sh + C::EPB * NV * NP;             // [EPB][NP]      squared sound speed
  double* fbuf = c2sh + C::EPB * NP;                  // [EPB][4][NF][NV]

  const int tid = threadIdx.x;
  const int el = tid / NF, t2 = tid % NF, i = t2 % Nq, j = t2 / Nq;
  const int e = blockIdx.x * C::EPB + el;
  const bool active = e < p.Ne;
  if (tid < Nq * Nq) Dsh[tid] = p.D[tid / Nq][tid % Nq];

  double* f1 = F1sh + el * NV * NP;
  double* f2 = F2sh + el * NV * NP;
  double* c2s = c2sh + el * NP;
  double* fb = fbuf + el * 4 * NF * NV;

  double acc[Nq][NV];      // sum_d D_d Ft^d - (1/w_0) sum_faces r   at the Nq nodes of the column
  double buoy[Nq];         // (rho - rho_r) g
#pragma unroll
  for (int k = 0; k < Nq; ++k)
#pragma unroll
    for (int v = 0; v < NV; ++v) acc[k][v] = 0.0;

  const int* nbr = p.nbr + (size_t)(active ? e : 0) * 6;
  if (active) {
#pragma unroll
    for (int k = 0; k < Nq; ++k) {
      const int n = t2 + NF * k;
      const size_t idx = (size_t)e * NP + n;
      double Y[6], g[12]; CmSite st; CmPrim P;
      cm_load_state<NV>(p.Q, p.stride, idx, Y);
      if (p.sgs) cm_load_state<NG>(p.G, p.stride, idx, g);
      cm_load_site<Nq, MOIST, GEOM>(p, e, n, k, st);
      cm_eos<MOIST>(p, Y, st, P);
      buoy[k] = P.drho * p.th.grav;
      double Fa[6], Fb[6], Fc[6];
      if constexpr (GEOM == 0) {
        cm_flux_axis<MOIST, 0>(Y, P, p.sgs, g, p.cA[0], Fa);
        cm_flux_axis<MOIST, 1>(Y, P, p.sgs, g, p.cA[1], Fb);
        cm_flux_axis<MOIST, 2>(Y, P, p.sgs, g, p.cA[2], Fc);
      } else {
        double Ja[9];
#pragma unroll
        for (int m = 0; m < 9; ++m) Ja[m] = __ldg(p.geo + (size_t)m * p.stride + idx);
        cm_flux_dir<MOIST>(Y, P, p.sgs, g, Ja[0], Ja[1], Ja[2], Fa);
        cm_flux_dir<MOIST>(Y, P, p.sgs, g, Ja[3], Ja[4], Ja[5], Fb);
        cm_flux_dir<MOIST>(Y, P, p.sgs, g, Ja[6], Ja[7], Ja[8], Fc);
      }
#pragma unroll
      for (int v = 0; v < NV; ++v) { f1[v * NP + n] = Fa[v]; f2[v * NP + n] = Fb[v]; }
      c2s[n] = P.c2;
      // zeta contraction in registers: acc[k'] += D[k'][k] Ft^3(k)
#pragma unroll
      for (int kk = 0; kk < Nq; ++kk)
#pragma unroll
        for (int v = 0; v < NV; ++v) acc[kk][v] += p.D[kk][k] * Fc[v];
      // zeta faces of this column
      if (k == 0 || k == N) {
        const int f = (k == 0) ? 4 : 5;
        double Ftm[6], r[6];
#pragma unroll
        for (int v = 0; v < NV; ++v) Ftm[v] = (k == 0) ? -Fc[v] : Fc[v];
        cm_tend_face<Nq, MOIST, GEOM>(p, e, __ldg(nbr + f), f, n, t2 + NF * (N - k), N - k, Y, Ftm, P.c2, r);
#pragma unroll
        for (int v = 0; v < NV; ++v) acc[k][v] -= p.inv_w0 * r[v];
      }
    }
  }
  __syncthreads();
  double Di[Nq], Dj[Nq];
#pragma unroll
  for (int m = 0; m < Nq; ++m) { Di[m] = Dsh[i * Nq + m]; Dj[m] = Dsh[j * Nq + m]; }

  if (active) {
    // lateral faces: node (a, b) = (i, j) of faces 0..3
#pragma unroll
    for (int f = 0; f < 4; ++f) {
      const int d = f >> 1;
      const int at = (f & 1) ? N : 0, ot = N - at;
      const int nm = (d == 0) ? (at + Nq * i + NF * j) : (i + Nq * at + NF * j);
      const int np_ = (d == 0) ? (ot + Nq * i + NF * j) : (i + Nq * ot + NF * j);
      double Ym[6], Ftm[6], r[6];
      cm_load_state<NV>(p.Q, p.stride, (size_t)e * NP + nm, Ym);
      const double* fs = (d == 0) ? f1 : f2;
#pragma unroll
      for (int v = 0; v < NV; ++v) Ftm[v] = (f & 1) ? fs[v * NP + nm] : -fs[v * NP + nm];
      cm_tend_face<Nq, MOIST, GEOM>(p, e, __ldg(nbr + f), f, nm, np_, j, Ym, Ftm, c2s[nm], r);
#pragma unroll
      for (int v = 0; v < NV; ++v) fb[(f * NF + t2) * NV + v] = r[v];
    }
    // xi / eta contractions from the staged tile
#pragma unroll
    for (int k = 0; k < Nq; ++k)
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        double a = 0.0;
#pragma unroll
        for (int m = 0; m < Nq; ++m)
          a += Di[m] * f1[v * NP + m + Nq * j + NF * k] + Dj[m] * f2[v * NP + i + Nq * m + NF * k];
        acc[k][v] += a;
      }
  }
  __syncthreads();
  if (!active) return;

#pragma unroll
  for (int k = 0; k < Nq; ++k) {
    const int n = t2 + NF * k;
    const size_t idx = (size_t)e * NP + n;
    const double invJ = (GEOM == 0) ? p.invJ : __ldg(p.geo + 9 * p.stride + idx);
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      double a = acc[k][v];
      if (i == 0) a -= p.inv_w0 * fb[(0 * NF + j + Nq * k) * NV + v];
      if (i == N) a -= p.inv_w0 * fb[(1 * NF + j + Nq * k) * NV + v];
      if (j == 0) a -= p.inv_w0 * fb[(2 * NF + i + Nq * k) * NV + v];
      if (j == N) a -= p.inv_w0 * fb[(3 * NF + i + Nq * k) * NV + v];
      double rhs = -invJ * a;
      if (v == 3) rhs -= buoy[k];                                     // -(rho - rho_r) grad Phi   (eq. 4)
      if (p.mode == 0) {
        p.dQ[v * p.stride + idx] = rhs;
      } else {
        // a5: dU <- A_s dU + dt RHS ; U <- U + B_s dU
        const double dold = (p.rka != 0.0) ? p.dQ[v * p.stride + idx] : 0.0;
        const double dnew = p.rka * dold + p.dt * rhs;
        p.dQ[v * p.stride + idx] = dnew;
        p.Qnew[v * p.stride + idx] = __ldg(p.Q + v * p.stride + idx) + p.rkb * dnew;
      }
    }
  }
}
