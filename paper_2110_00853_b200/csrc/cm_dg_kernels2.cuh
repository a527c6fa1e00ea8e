// cm_dg_kernels2.cuh -- thread-per-node kernels for ANY geometry (stored metric terms, per-node reference state): the
// path of warped meshes (geom != 0) and of reference states that are not columns; on flat bricks the row-sweep /
// CTA-per-element kernels are used instead (cm_dg_tuning.kernel = 2 forces these).
//   * one thread owns ONE node, a CTA holds EPB elements x TPE threads (~64-100 registers per thread, several CTAs per
//     SM): latency is hidden by thread-level parallelism;
//   * the tensor-product contractions are done by LINE tasks: a thread owns one xi/eta/zeta line of one element,
//     reads its Nq values from shared memory, applies the full Nq x Nq matrix with D as constant-bank operands
//     (no D registers) and writes the Nq results back (in place for the divergence);
//   * face work is a list of 6*Nq^2 FACE tasks per element spread evenly over the CTA's threads; a face whose
//     neighbour element lives in the same CTA reads the neighbour's state and contravariant flux straight from
//     shared memory (no global loads, no second EOS / flux evaluation); only CTA-external faces go to L2.
// On stored-metric meshes the tendency kernel of cm_dg_kernels11.cuh (CTA per element, bulk-TMA staging) is the default
// and this file serves the gradient, the HLLC / Roe fluxes and the saturation-adjusted equation of state; kernel = 2 selects
// the tendency kernel below as well.  Both kernels prefetch the arrays of the element one wave of CTAs ahead into L2.
// Parity-tested on all five configs; profile: profiles/r2_stored_metric.md.  P:L<n> = paper line.
#pragma once
#include "cm_dg_internal.h"
#include "cm_dg_physics.cuh"

template <int Nq> struct CmCfg2 {
  static constexpr int NF = Nq * Nq;
  static constexpr int NP = Nq * Nq * Nq;
  static constexpr int TPE = ((NP + 31) / 32) * 32;                 // threads per element
  static constexpr int EPB = (Nq <= 3) ? 8 : (Nq == 4) ? 4 : (Nq == 5) ? 2 : 1;
  static constexpr int THREADS = EPB * TPE;
  static constexpr int MINB = (Nq <= 5) ? 3 : (Nq == 6) ? 3 : (Nq == 7) ? 2 : 1;   // CTAs per SM the register budget aims at
#ifndef CM_2_MINB_T
#define CM_2_MINB_T MINB
#endif
  static constexpr int MINB_T = CM_2_MINB_T;       // same for the tendency kernel
};

// L2 prefetch of the n doubles at a (cp.async.bulk.prefetch.L2 wants a 16-byte aligned address and size; the state arrays
// are padded by one double, so rounding outwards stays inside them)
__device__ __forceinline__ void cm2_prefetch_tile(const double* a, int n) {
  const unsigned long long lo = (unsigned long long)a & ~15ull, hi = ((unsigned long long)(a + n) + 15ull) & ~15ull;
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(lo), "r"((unsigned)(hi - lo)) : "memory");
}
// every array the kernels will read for element ea (one wave of resident CTAs further on in the launch order) into L2, one
// tile per thread t: the loads of that CTA then wait on L2, not on DRAM
template <int NP, int GEOM>
__device__ __forceinline__ void cm2_prefetch_element(const CmKP& p, int ea, int t, int nv, bool with_g, int ng, bool with_res) {
  if (ea >= p.Ne) return;
  const size_t off = (size_t)ea * NP;
  int k = t;
  if (k < nv) { cm2_prefetch_tile(p.Q + (size_t)k * p.stride + off, NP); return; }
  k -= nv;
  if (with_g) { if (k < ng) { cm2_prefetch_tile(p.G + (size_t)k * p.stride + off, NP); return; } k -= ng; }
  if (with_res) { if (k < nv) { cm2_prefetch_tile(p.dQ + (size_t)k * p.stride + off, NP); return; } k -= nv; }
  if (GEOM != 0) {
    if (k < CM_NGEO) { cm2_prefetch_tile(p.geo + (size_t)k * p.stride + off, NP); return; }
    k -= CM_NGEO;
    if (p.use_ref && k < 3 && (k < 2 || nv == 6)) cm2_prefetch_tile(p.ref + (size_t)k * p.stride + off, NP);
  }
}

// node indices of face task (f, a, b): own node nm, coincident node np_ of the neighbour, their zeta indices
template <int Nq>
__device__ __forceinline__ void cm2_face_nodes(int f, int a, int b, int& nm, int& np_, int& km, int& kp) {
  constexpr int N = Nq - 1, NF = Nq * Nq;
  const int d = f >> 1;
  const int at = (f & 1) ? N : 0, ot = N - at;
  if (d == 0) { nm = at + Nq * a + NF * b; np_ = ot + Nq * a + NF * b; km = b; kp = b; }
  else if (d == 1) { nm = a + Nq * at + NF * b; np_ = a + Nq * ot + NF * b; km = b; kp = b; }
  else { nm = a + Nq * b + NF * at; np_ = a + Nq * b + NF * ot; km = at; kp = ot; }
}

// ------------------------------------------------------------------------------------------------
// a2: auxiliary gradient + Smagorinsky-Lilly, thread per node
// ------------------------------------------------------------------------------------------------
// RICH: theta_v is a further gradient variable (eq. 40)
template <int Nq, bool MOIST, int GEOM, bool RICH = false, bool SAT = false>
__global__ void __launch_bounds__(CmCfg2<Nq>::THREADS, CmCfg2<Nq>::MINB) cm2_gradient_kernel(const __grid_constant__ CmKP p) {
  using C = CmCfg2<Nq>;
  constexpr int NF = C::NF, NP = C::NP, N = Nq - 1, TPE = C::TPE, EPB = C::EPB;
  constexpr int NV = MOIST ? 6 : 5;
  constexpr int NS0 = MOIST ? 5 : 4;                   // u, v, w, h_tot, [q_t]
  constexpr int NS = NS0 + (RICH ? 1 : 0);             // + theta_v
  extern __shared__ double smem[];
  double* s_sh = smem;                               // [EPB][NS][NP]      gradient variables
  double* d_sh = s_sh + EPB * NS * NP;               // [3][EPB][NS][NP]   reference-space derivatives
  double* fbuf = d_sh + 3 * EPB * NS * NP;           // [EPB][6*NF][NS]    s* - s^- per face node

  const int tid = threadIdx.x;
  const int el = tid / TPE, t = tid % TPE;
  const int e0 = blockIdx.x * EPB;
  const int e = e0 + el;
  const bool active = e < p.Ne;
  if (p.ahead > 0 && active) cm2_prefetch_element<NP, GEOM>(p, e + p.ahead, t, NV, false, 0, false);

  if (active && t < NP) {
    double Y[6]; CmSite st; CmPrim P;
    cm_load_state<NV>(p.Q, p.stride, (size_t)e * NP + t, Y);
    cm_load_site<Nq, MOIST, GEOM>(p, e, t, t / NF, st);
    cm_eos<MOIST, SAT>(p, Y, st, P);
    double* s = s_sh + (size_t)el * NS * NP + t;
    s[0] = P.u; s[NP] = P.v; s[2 * NP] = P.w; s[3 * NP] = P.h;
    if (MOIST) s[4 * NP] = P.q;
    if (RICH) s[NS0 * NP] = cm_theta_v(p.th, P.p, P.ir);
  }
  __syncthreads();

  if (active) {
    // line tasks: d(s)/d(xi_d) along one line, all variables
    for (int lt = t; lt < 3 * NF; lt += TPE) {
      const int d = lt / NF, l = lt % NF;
      const int base = (d == 0) ? Nq * l : (d == 1) ? (l % Nq) + NF * (l / Nq) : l;
      const int str = (d == 0) ? 1 : (d == 1) ? Nq : NF;
#pragma unroll
      for (int v = 0; v < NS; ++v) {
        const double* in = s_sh + ((size_t)el * NS + v) * NP + base;
        double* out = d_sh + (((size_t)d * EPB + el) * NS + v) * NP + base;
        double x[Nq];
#pragma unroll
        for (int m = 0; m < Nq; ++m) x[m] = in[m * str];
#pragma unroll
        for (int i = 0; i < Nq; ++i) {
          double a = 0.0;
#pragma unroll
          for (int m = 0; m < Nq; ++m) a += p.D[i][m] * x[m];
          out[i * str] = a;
        }
      }
    }
    // face tasks
    for (int ft = t; ft < 6 * NF; ft += TPE) {
      const int f = ft / NF, idx = ft % NF;
      int nm, np_, km, kp;
      cm2_face_nodes<Nq>(f, idx % Nq, idx / Nq, nm, np_, km, kp);
      const int d = f >> 1;
      const double sgn = (f & 1) ? 1.0 : -1.0;
      const int nb = __ldg(p.nbr + (size_t)e * 6 + f);
      double sm[6], delta[6];
#pragma unroll
      for (int v = 0; v < NS; ++v) sm[v] = s_sh[((size_t)el * NS + v) * NP + nm];
      if (nb >= e0 && nb < e0 + EPB) {
        const double* sp = s_sh + (size_t)(nb - e0) * NS * NP + np_;
#pragma unroll
        for (int v = 0; v < NS; ++v) delta[v] = 0.5 * (sp[v * NP] - sm[v]);
      } else if (nb >= 0) {
        double Y[6]; CmSite st; CmPrim P;
        cm_load_state<NV>(p.Q, p.stride, (size_t)nb * NP + np_, Y);
        cm_load_site<Nq, MOIST, GEOM>(p, nb, np_, kp, st);
        cm_eos<MOIST, SAT>(p, Y, st, P);
        delta[0] = 0.5 * (P.u - sm[0]); delta[1] = 0.5 * (P.v - sm[1]); delta[2] = 0.5 * (P.w - sm[2]);
        delta[3] = 0.5 * (P.h - sm[3]);
        if (MOIST) delta[4] = 0.5 * (P.q - sm[4]);
        if (RICH) delta[NS0] = 0.5 * (cm_theta_v(p.th, P.p, P.ir) - sm[NS0]);
      } else {
        // wall: u_bc = u^- - (n.u^-) n  (A6); scalars unchanged (A8)
        double A[3]; cm_face_vector<Nq, GEOM>(p, e, nm, d, sgn, A);
        const double ua = (sm[0] * A[0] + sm[1] * A[1] + sm[2] * A[2]) / (A[0] * A[0] + A[1] * A[1] + A[2] * A[2]);
        delta[0] = -ua * A[0]; delta[1] = -ua * A[1]; delta[2] = -ua * A[2]; delta[3] = 0.0; delta[4] = 0.0; delta[5] = 0.0;
      }
      double* fb = fbuf + ((size_t)el * 6 * NF + ft) * NS;
#pragma unroll
      for (int v = 0; v < NS; ++v) fb[v] = delta[v];
    }
  }
  __syncthreads();
  if (!active || t >= NP) return;

  const int n = t, i = n % Nq, j = (n / Nq) % Nq, k = n / NF;
  const size_t idx = (size_t)e * NP + n;
  double Ja[3][3], invJ, cs2d2, d2x, d2y, d2z;
  if constexpr (GEOM == 0) {
    invJ = p.invJ; cs2d2 = p.cs2delta2; d2x = p.d2[0]; d2y = p.d2[1]; d2z = p.d2[2];
  } else {
#pragma unroll
    for (int d = 0; d < 3; ++d)
#pragma unroll
      for (int c = 0; c < 3; ++c) Ja[d][c] = __ldg(p.geo + (size_t)(3 * d + c) * p.stride + idx);
    invJ = __ldg(p.geo + 9 * p.stride + idx);
    cs2d2 = __ldg(p.geo + 11 * p.stride + idx);
    d2x = __ldg(p.geo + 12 * p.stride + idx); d2y = __ldg(p.geo + 13 * p.stride + idx); d2z = __ldg(p.geo + 14 * p.stride + idx);
  }
  const double* fb = fbuf + (size_t)el * 6 * NF * NS;
  const double w0i = p.inv_w0;
  double G[6][3];
#pragma unroll
  for (int v = 0; v < NS; ++v) {
    double dr = d_sh[(((size_t)0 * EPB + el) * NS + v) * NP + n];
    double ds = d_sh[(((size_t)1 * EPB + el) * NS + v) * NP + n];
    double dt = d_sh[(((size_t)2 * EPB + el) * NS + v) * NP + n];
    if (i == 0) dr -= w0i * fb[(0 * NF + j + Nq * k) * NS + v];
    if (i == N) dr += w0i * fb[(1 * NF + j + Nq * k) * NS + v];
    if (j == 0) ds -= w0i * fb[(2 * NF + i + Nq * k) * NS + v];
    if (j == N) ds += w0i * fb[(3 * NF + i + Nq * k) * NS + v];
    if (k == 0) dt -= w0i * fb[(4 * NF + i + Nq * j) * NS + v];
    if (k == N) dt += w0i * fb[(5 * NF + i + Nq * j) * NS + v];
    if constexpr (GEOM == 0) {
      G[v][0] = (p.cA[0] * invJ) * dr; G[v][1] = (p.cA[1] * invJ) * ds; G[v][2] = (p.cA[2] * invJ) * dt;
    } else {
#pragma unroll
      for (int c = 0; c < 3; ++c) G[v][c] = invJ * (Ja[0][c] * dr + Ja[1][c] * ds + Ja[2][c] * dt);
    }
  }
  if (!MOIST) { if (RICH) { G[5][2] = G[4][2]; } G[4][0] = G[4][1] = G[4][2] = 0.0; }   // dry: theta_v sits in slot 4
  if (p.mode == 1) {
#pragma unroll
    for (int v = 0; v < 5; ++v)
#pragma unroll
      for (int c = 0; c < 3; ++c) p.Gout[(size_t)(3 * v + c) * p.stride + idx] = G[v][c];
  } else {
    // eq. (33)-(40): closure (cm_closure); store tau, J + D, d_q
    double Gr[5][3];
#pragma unroll
    for (int v = 0; v < 5; ++v)
#pragma unroll
      for (int c = 0; c < 3; ++c) Gr[v][c] = G[v][c];
    double thv = 1.0, dthv = 0.0;
    if (RICH) { thv = s_sh[((size_t)el * NS + NS0) * NP + n]; dthv = G[5][2]; }
    double g[12];
    cm_closure<MOIST>(p, Gr, cs2d2, d2x, d2y, d2z, thv, dthv, g);
    double* o = p.Gout + idx;
#pragma unroll
    for (int kk = 0; kk < (MOIST ? 12 : 9); ++kk) o[kk * p.stride] = g[kk];
  }
}

// ------------------------------------------------------------------------------------------------
// a3-a5: tendency + fused LSRK update, thread per node
// ------------------------------------------------------------------------------------------------
template <int Nq, bool MOIST, int GEOM, bool SAT = false>
__global__ void __launch_bounds__(CmCfg2<Nq>::THREADS, CmCfg2<Nq>::MINB_T) cm2_tendency_kernel(const __grid_constant__ CmKP p) {
  using C = CmCfg2<Nq>;
  constexpr int NF = C::NF, NP = C::NP, N = Nq - 1, TPE = C::TPE, EPB = C::EPB;
  constexpr int NV = MOIST ? 6 : 5;
  constexpr int NG = MOIST ? 12 : 9;
  extern __shared__ double smem[];
  double* Q_sh = smem;                               // [EPB][NV][NP]     state
  double* F_sh = Q_sh + EPB * NV * NP;               // [3][EPB][NV][NP]  contravariant fluxes, then D_d Ft^d in place
  double* c2sh = F_sh + 3 * EPB * NV * NP;           // [EPB][NP]         squared sound speed
  double* fbuf = c2sh + EPB * NP;                    // [EPB][6*NF][NV]   sgn*Ft^- - sJ F* per face node

  const int tid = threadIdx.x;
  const int el = tid / TPE, t = tid % TPE;
  const int e0 = blockIdx.x * EPB;
  const int e = e0 + el;
  const bool active = e < p.Ne;
  if (p.ahead > 0 && active) cm2_prefetch_element<NP, GEOM>(p, e + p.ahead, t, NV, p.sgs != 0, NG, p.mode == 1 && p.rka != 0.0);
  double buoy = 0.0, taus = 0.0;

  // ---- phase 0: primitives and fluxes of the own node -> shared memory
  if (active && t < NP) {
    const size_t idx = (size_t)e * NP + t;
    double Y[6], g[12]; CmSite st; CmPrim P;
    cm_load_state<NV>(p.Q, p.stride, idx, Y);
    if (p.sgs) cm_load_state<NG>(p.G, p.stride, idx, g);
    cm_load_site<Nq, MOIST, GEOM>(p, e, t, t / NF, st);
    cm_eos<MOIST, SAT>(p, Y, st, P);
    buoy = P.drho * p.th.grav; taus = st.taus;
    double* q = Q_sh + (size_t)el * NV * NP + t;
#pragma unroll
    for (int v = 0; v < NV; ++v) q[v * NP] = Y[v];
    c2sh[el * NP + t] = P.c2;
    double Fa[6];
    double* f0 = F_sh + ((size_t)(0 * EPB + el) * NV) * NP + t;
    double* f1 = F_sh + ((size_t)(1 * EPB + el) * NV) * NP + t;
    double* f2 = F_sh + ((size_t)(2 * EPB + el) * NV) * NP + t;
    if constexpr (GEOM == 0) {
      cm_flux_axis<MOIST, 0>(Y, P, p.sgs, g, p.cA[0], Fa);
#pragma unroll
      for (int v = 0; v < NV; ++v) f0[v * NP] = Fa[v];
      cm_flux_axis<MOIST, 1>(Y, P, p.sgs, g, p.cA[1], Fa);
#pragma unroll
      for (int v = 0; v < NV; ++v) f1[v * NP] = Fa[v];
      cm_flux_axis<MOIST, 2>(Y, P, p.sgs, g, p.cA[2], Fa);
#pragma unroll
      for (int v = 0; v < NV; ++v) f2[v * NP] = Fa[v];
    } else {
      double Ja[9];
#pragma unroll
      for (int m = 0; m < 9; ++m) Ja[m] = __ldg(p.geo + (size_t)m * p.stride + idx);
      cm_flux_dir<MOIST>(Y, P, p.sgs, g, Ja[0], Ja[1], Ja[2], Fa);
#pragma unroll
      for (int v = 0; v < NV; ++v) f0[v * NP] = Fa[v];
      cm_flux_dir<MOIST>(Y, P, p.sgs, g, Ja[3], Ja[4], Ja[5], Fa);
#pragma unroll
      for (int v = 0; v < NV; ++v) f1[v * NP] = Fa[v];
      cm_flux_dir<MOIST>(Y, P, p.sgs, g, Ja[6], Ja[7], Ja[8], Fa);
#pragma unroll
      for (int v = 0; v < NV; ++v) f2[v * NP] = Fa[v];
    }
  }
  __syncthreads();

  // ---- phase 1: face tasks (read the untouched fluxes at face nodes)
  if (active) {
    for (int ft = t; ft < 6 * NF; ft += TPE) {
      const int f = ft / NF, fi = ft % NF;
      int nm, np_, km, kp;
      cm2_face_nodes<Nq>(f, fi % Nq, fi / Nq, nm, np_, km, kp);
      const int d = f >> 1;
      const double sgn = (f & 1) ? 1.0 : -1.0;
      const int nb = __ldg(p.nbr + (size_t)e * 6 + f);
      double A[3]; cm_face_vector<Nq, GEOM>(p, e, nm, d, sgn, A);
      const double sJ = (GEOM == 0) ? p.cA[d] : sqrt(A[0] * A[0] + A[1] * A[1] + A[2] * A[2]);
      double Ym[6], Ftm[6], r[6];
      const double* qm = Q_sh + (size_t)el * NV * NP + nm;
      const double* fm = F_sh + ((size_t)(d * EPB + el) * NV) * NP + nm;
#pragma unroll
      for (int v = 0; v < NV; ++v) { Ym[v] = qm[v * NP]; Ftm[v] = sgn * fm[v * NP]; }
      const double c2m = c2sh[el * NP + nm];
      const double uAm = (Ym[1] * A[0] + Ym[2] * A[1] + Ym[3] * A[2]) * cm_rcp(Ym[0]);   // sJ (u^- . n)
      const double cm_ = cm_sqrt(c2m);
      if (nb >= 0) {
        double Yp[6], Fp[6], c2p, uAp;
        if (nb >= e0 && nb < e0 + EPB) {
          // neighbour element is in this CTA: its state and contravariant flux are already in shared memory;
          // the face vectors of the two sides are equal and opposite, so A . F^+ = sgn * Ft^d(neighbour node)
          const int eln = nb - e0;
          const double* qp = Q_sh + (size_t)eln * NV * NP + np_;
          const double* fp = F_sh + ((size_t)(d * EPB + eln) * NV) * NP + np_;
#pragma unroll
          for (int v = 0; v < NV; ++v) { Yp[v] = qp[v * NP]; Fp[v] = sgn * fp[v * NP]; }
          c2p = c2sh[eln * NP + np_];
          uAp = (Yp[1] * A[0] + Yp[2] * A[1] + Yp[3] * A[2]) * cm_rcp(Yp[0]);
        } else {
          double g[12]; CmSite st; CmPrim P;
          const size_t idp = (size_t)nb * NP + np_;
          cm_load_state<NV>(p.Q, p.stride, idp, Yp);
          if (p.sgs) cm_load_state<NG>(p.G, p.stride, idp, g);
          cm_load_site<Nq, MOIST, GEOM>(p, nb, np_, kp, st);
          cm_eos<MOIST, SAT>(p, Yp, st, P);
          cm_flux_dir<MOIST>(Yp, P, p.sgs, g, A[0], A[1], A[2], Fp);
          c2p = P.c2;
          uAp = A[0] * P.u + A[1] * P.v + A[2] * P.w;
        }
        if (p.riemann == 0) {
          const double lamsJ = fmax(fabs(uAm) + cm_ * sJ, fabs(uAp) + cm_sqrt(c2p) * sJ);   // sJ * lambda (R2)
#pragma unroll
          for (int v = 0; v < NV; ++v) r[v] = 0.5 * (Ftm[v] - Fp[v]) - 0.5 * lamsJ * (Ym[v] - Yp[v]);
        } else {
          // HLLC or Roe for F1, central flux for F2: sJ F* = Fs + (1/2)(Ftm - A.F1^-) + (1/2)(Fp - A.F1^+)
          CmSite sm_, sp_; CmPrim Pm, Pp; double AFm[6], AFp[6], Fs[6];
          cm_load_site<Nq, MOIST, GEOM>(p, e, nm, km, sm_); cm_eos<MOIST, SAT>(p, Ym, sm_, Pm);
          cm_load_site<Nq, MOIST, GEOM>(p, nb, np_, kp, sp_); cm_eos<MOIST, SAT>(p, Yp, sp_, Pp);
          cm_flux1_dir<MOIST>(Ym, Pm, A[0], A[1], A[2], AFm); cm_flux1_dir<MOIST>(Yp, Pp, A[0], A[1], A[2], AFp);
          if (p.riemann == 1) cm_hllc<MOIST>(Ym, Pm, AFm, Yp, Pp, AFp, A, sJ, Fs);
          else cm_roe<MOIST>(p, Ym, Pm, AFm, Yp, Pp, AFp, A, sJ, sm_.Phi, Fs);
#pragma unroll
          for (int v = 0; v < NV; ++v) r[v] = Ftm[v] - (Fs[v] + 0.5 * (Ftm[v] - AFm[v]) + 0.5 * (Fp[v] - AFp[v]));
        }
      } else {
        // free-slip wall (A6-A7): Rusanov against the mirrored state = [0; (p' + rho u_n (u_n + lambda)) n; 0; 0];
        // second-order normal fluxes vanish (R10) except the prescribed bottom energy flux
        CmSite st; CmPrim P;
        cm_load_site<Nq, MOIST, GEOM>(p, e, nm, km, st);
        cm_eos<MOIST, SAT>(p, Ym, st, P);
        const double un = uAm / sJ;
        if (p.riemann == 0) {
          const double lam = fabs(un) + cm_;
          const double mom = P.pp + Ym[0] * un * (un + lam);
#pragma unroll
          for (int v = 0; v < NV; ++v) r[v] = Ftm[v];
          r[1] -= mom * A[0]; r[2] -= mom * A[1]; r[3] -= mom * A[2];
        } else {
          // HLLC / Roe against the mirrored state (A6)-(A7); n.F2* = 0 at the wall (R10)
          double Yg[6], AFm[6], AFg[6], Fs[6];
          const double mn = 2.0 * (Ym[1] * A[0] + Ym[2] * A[1] + Ym[3] * A[2]) / (sJ * sJ);
#pragma unroll
          for (int v = 0; v < NV; ++v) Yg[v] = Ym[v];
          Yg[1] -= mn * A[0]; Yg[2] -= mn * A[1]; Yg[3] -= mn * A[2];
          CmPrim Pg = P;
          Pg.u = Yg[1] * P.ir; Pg.v = Yg[2] * P.ir; Pg.w = Yg[3] * P.ir;
          cm_flux1_dir<MOIST>(Ym, P, A[0], A[1], A[2], AFm); cm_flux1_dir<MOIST>(Yg, Pg, A[0], A[1], A[2], AFg);
          if (p.riemann == 1) cm_hllc<MOIST>(Ym, P, AFm, Yg, Pg, AFg, A, sJ, Fs);
          else cm_roe<MOIST>(p, Ym, P, AFm, Yg, Pg, AFg, A, sJ, st.Phi, Fs);
#pragma unroll
          for (int v = 0; v < NV; ++v) r[v] = Ftm[v] - Fs[v];
        }
        if (f == 4) cm_surface_flux<MOIST>(p, A, sJ, Ym[0], qm + NF, NP, r);   // the node above nm: first interior layer
      }
      double* fb = fbuf + ((size_t)el * 6 * NF + ft) * NV;
#pragma unroll
      for (int v = 0; v < NV; ++v) fb[v] = r[v];
    }
  }
  __syncthreads();

  // ---- phase 2: line tasks, Ft^d <- D_d Ft^d in place
  if (active) {
    for (int lt = t; lt < 3 * NF; lt += TPE) {
      const int d = lt / NF, l = lt % NF;
      const int base = (d == 0) ? Nq * l : (d == 1) ? (l % Nq) + NF * (l / Nq) : l;
      const int str = (d == 0) ? 1 : (d == 1) ? Nq : NF;
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        double* a = F_sh + ((size_t)(d * EPB + el) * NV + v) * NP + base;
        double x[Nq], y[Nq];
#pragma unroll
        for (int m = 0; m < Nq; ++m) x[m] = a[m * str];
#pragma unroll
        for (int i = 0; i < Nq; ++i) {
          double s = 0.0;
#pragma unroll
          for (int m = 0; m < Nq; ++m) s += p.D[i][m] * x[m];
          y[i] = s;
        }
#pragma unroll
        for (int i = 0; i < Nq; ++i) a[i * str] = y[i];
      }
    }
  }
  __syncthreads();
  if (!active || t >= NP) return;

  // ---- phase 3: assemble the tendency of the own node and update
  const int n = t, i = n % Nq, j = (n / Nq) % Nq, k = n / NF;
  const size_t idx = (size_t)e * NP + n;
  const double invJ = (GEOM == 0) ? p.invJ : __ldg(p.geo + 9 * p.stride + idx);
  double dold[6];
  const bool stage = (p.mode != 0);
  const bool readres = stage && (p.rka != 0.0);
#pragma unroll
  for (int v = 0; v < NV; ++v) dold[v] = readres ? p.dQ[v * p.stride + idx] : 0.0;
  const double* fb = fbuf + (size_t)el * 6 * NF * NV;
#pragma unroll
  for (int v = 0; v < NV; ++v) {
    double a = F_sh[((size_t)(0 * EPB + el) * NV + v) * NP + n] + F_sh[((size_t)(1 * EPB + el) * NV + v) * NP + n] +
               F_sh[((size_t)(2 * EPB + el) * NV + v) * NP + n];
    double fs = 0.0;
    if (i == 0) fs += fb[(0 * NF + j + Nq * k) * NV + v];
    if (i == N) fs += fb[(1 * NF + j + Nq * k) * NV + v];
    if (j == 0) fs += fb[(2 * NF + i + Nq * k) * NV + v];
    if (j == N) fs += fb[(3 * NF + i + Nq * k) * NV + v];
    if (k == 0) fs += fb[(4 * NF + i + Nq * j) * NV + v];
    if (k == N) fs += fb[(5 * NF + i + Nq * j) * NV + v];
    double rhs = -invJ * (a - p.inv_w0 * fs);
    if (v == 3) rhs -= buoy;                                     // -(rho - rho_r) grad Phi   (eq. 4)
    if (v >= 1 && v <= 3)                                        // Rayleigh sponge (A4); tau_s = 0 outside the layer
      rhs -= taus * (Q_sh[((size_t)el * NV + v) * NP + n] - Q_sh[((size_t)el * NV) * NP + n] * p.urelax[v - 1]);
    if (!stage) {
      p.dQ[v * p.stride + idx] = rhs;
    } else {
      // a5: dU <- A_s dU + dt RHS ; U <- U + B_s dU
      const double dnew = p.rka * dold[v] + p.dt * rhs;
      p.dQ[v * p.stride + idx] = dnew;
      p.Qnew[v * p.stride + idx] = Q_sh[((size_t)el * NV + v) * NP + n] + p.rkb * dnew;
    }
  }
}
