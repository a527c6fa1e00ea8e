// cm_dg_kernels5.cuh -- the hot kernels for flat bricks (GEOM == 0): one small CTA per element, own data by bulk
// TMA, thread per node, fused line + face tasks.
//
// What the earlier variants taught (profiles/r1a_v2.md, profiles/r1b_v4.md): every variant issued one warp
// instruction per 15-19 cycles per warp, 40-60 % of it `long_scoreboard`: a thread waits ~1000 cycles on a global
// load several dozen times per element (own nodes, neighbour traces, residual, spill reloads), and neither
// 24 barrier-coupled warps (v2) nor 9 free-running warps with 4 nodes per lane (v4) hide that.  Here
//   * ONE elected thread fetches the element's own Q, packed SGS fluxes G and LSRK residual with 1-D bulk TMA
//     (cp.async.bulk ... mbarrier::complete_tx) into shared memory the moment the CTA starts: no thread ever waits
//     on a global load of own data, no register holds a prefetched value, and there is ONE wait (an mbarrier) per
//     element.  A tile is NP*8 bytes; for odd NP it is fetched as NP+1 doubles from the 16-byte boundary below it,
//     so the data sit at offset (e & 1) of the slot;
//   * the CTA is small (NP threads rounded to warps, one node per thread, ~30 KB of shared memory at N = 4) so six
//     of them are resident per SM and run out of phase: while one waits for its tiles the others compute;
//   * phase 1 (thread per node): EOS + contravariant fluxes, F^1, F^2 overwrite the G slots in place;
//   * phase 2 (thread per line, one warp per direction): D_d F^d along the line in registers (D from the constant
//     bank) and the numerical flux at the line's two end nodes (neighbour trace gathered from L2: 6 + 5 values),
//     lifted and folded into the end values before the line is written back -- no face buffers, no second pass;
//   * phase 3 (thread per node): sum of the three directions, gravity source, fused LSRK update, coalesced stores.
// Two CTA barriers per element.  Arithmetic follows cm_dg_physics.cuh.  P:L<n> = paper line.
#pragma once
#include "cm_dg_internal.h"
#include "cm_dg_physics.cuh"

// ------------------------------------------------------------------------------------------------ PTX helpers
__device__ __forceinline__ uint32_t cm5_saddr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cm5_mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(cm5_saddr(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void cm5_mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(cm5_saddr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cm5_mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "LAB_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra LAB_WAIT;\n"
      "DONE:\n"
      "}\n" ::"r"(cm5_saddr(bar)), "r"(parity) : "memory");
}
// 1-D bulk TMA global -> shared, completion counted in bytes on an mbarrier (16-byte aligned src, dst, size)
__device__ __forceinline__ void cm5_bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(cm5_saddr(dst)),
               "l"(src), "r"(bytes), "r"(cm5_saddr(bar)) : "memory");
}
__device__ __forceinline__ void cm5_fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

template <int Nq, bool MOIST> struct CmCfg5 {
  static constexpr int NF = Nq * Nq;
  static constexpr int NP = Nq * Nq * Nq;
  static constexpr int NV = MOIST ? 6 : 5;
  static constexpr int NG = MOIST ? 12 : 9;
  static constexpr int NS = MOIST ? 5 : 4;                  // gradient variables u, v, w, h_tot, [q]
  static constexpr int NGD = MOIST ? 5 : 4;                 // SGS values one face direction needs
  static constexpr int ODD = NP & 1;
  static constexpr int SLOT = NP + ODD;                     // doubles per field tile in shared memory (16-byte multiple)
  static constexpr int THREADS = ((NP + 31) / 32) * 32;
  static constexpr int NFP = ((NF + 31) / 32) * 32;         // line tasks of one direction, padded to whole warps
  static constexpr int GS = (NG > 2 * NV) ? NG : 2 * NV;    // G slots, reused for F^1, F^2
  static constexpr int TEND_DOUBLES = (NV + GS + NV + 1 + NV) * SLOT;     // Q, G/F12, F3, c, residual
  static constexpr int GRAD_DOUBLES = (NV + 3 * NS) * SLOT;               // Q (then s in place), ds/dxi_d
  static constexpr size_t TEND_SMEM = sizeof(double) * TEND_DOUBLES + 16;
  static constexpr size_t GRAD_SMEM = sizeof(double) * GRAD_DOUBLES + 16;
  static constexpr int fit(size_t smem) { return (int)(233472 / (smem + 1024)); }
  static constexpr int cap(int b, int hi) { return b < 1 ? 1 : (b > hi ? hi : b); }
  static constexpr int MINB_T = cap(fit(TEND_SMEM), cap(2048 / THREADS, 6));
  static constexpr int MINB_G = cap(fit(GRAD_SMEM), cap(2048 / THREADS, 8));
};

__device__ __forceinline__ void cm5_site(const CmKP& p, int row, CmSite& s) {
  const double2* t = reinterpret_cast<const double2*>(p.ztab + (size_t)row * CM_ZTAB_W);
  const double2 a = __ldg(t), b = __ldg(t + 1), c = __ldg(t + 2), d = __ldg(t + 3);
  s.Phi = a.x; s.rho_r = a.y; s.rhoe_r = b.x; s.rhoq_r = b.y; s.E_r = c.x; s.q_r = c.y; s.icvm_r = d.x;
}

// primitives the gradient needs (u, v, w, h_tot, q): eq. (6)-(10), (13)-(14)
template <bool MOIST>
__device__ __forceinline__ void cm5_eos_grad(const CmKP& p, const double* Y, double Phi, double* s) {
  const CmThermo& th = p.th;
  const double ir = cm_rcp(Y[0]);
  const double u = Y[1] * ir, v = Y[2] * ir, w = Y[3] * ir;
  const double rq = MOIST ? Y[5] : 0.0;
  const double q = MOIST ? rq * ir : 0.0;
  const double K = 0.5 * (Y[1] * u + Y[2] * v + Y[3] * w);
  double kappa;
  if (MOIST) kappa = (th.R_d + th.a * q) * cm_rcp(th.c_vd + th.b * q); else kappa = th.kappa_d;
  const double E = Y[4] - K - Y[0] * Phi - rq * th.I_v0;
  const double pr = kappa * E + th.T_0 * (th.R_d * Y[0] + th.a * rq);
  s[0] = u; s[1] = v; s[2] = w; s[3] = (Y[4] + pr) * ir; s[4] = q;
}

// index into the packed SGS array (tau xx,yy,zz,xy,xz,yz | J+D x,y,z | d_q x,y,z) of the k-th value axis d needs
__host__ __device__ constexpr int cm5_gidx(int d, int k) {
  return (k == 3) ? 6 + d : (k == 4) ? 9 + d : (k == d) ? d : k + d + 2;   // (0,1)->3, (0,2)->4, (1,2)->5
}

// contravariant flux along axis D, A = s * e_D; gd = the SGS values that axis needs: tau(D,0..2), (J+D)_D, [d_q,D]
template <bool MOIST, bool SGS, int D>
__device__ __forceinline__ void cm5_flux_face(const double* Y, const CmPrim& P, const double* gd, double s, double* Fn) {
  const double ud = (D == 0) ? P.u : (D == 1) ? P.v : P.w;
  double wA = ud, t0 = 0.0, t1 = 0.0, t2 = 0.0, eA = 0.0, dqA = 0.0;
  if (SGS) {
    t0 = gd[0]; t1 = gd[1]; t2 = gd[2];
    eA = t0 * P.u + t1 * P.v + t2 * P.w + gd[3];
    if (MOIST) { dqA = gd[4]; wA += dqA; }
  }
  Fn[0] = s * (Y[0] * wA);
  Fn[1] = s * (Y[1] * wA + ((D == 0) ? P.pp : 0.0) + Y[0] * t0);
  Fn[2] = s * (Y[2] * wA + ((D == 1) ? P.pp : 0.0) + Y[0] * t1);
  Fn[3] = s * (Y[3] * wA + ((D == 2) ? P.pp : 0.0) + Y[0] * t2);
  Fn[4] = s * ((Y[4] + P.p) * ud + Y[0] * eA);
  if (MOIST) Fn[5] = s * (Y[5] * ud + Y[0] * dqA);
}

template <int Nq, int D> struct Cm5Str { static constexpr int value = (D == 0) ? 1 : (D == 1) ? Nq : Nq * Nq; };
// first node of line l of direction D, and the zeta index of the line (D < 2)
template <int Nq, int D>
__device__ __forceinline__ void cm5_line(int l, int& base, int& kline) {
  constexpr int NF = Nq * Nq;
  const int a = l % Nq, b = l / Nq;
  base = (D == 0) ? Nq * l : (D == 1) ? a + NF * b : l;
  kline = b;
}

// ------------------------------------------------------------------------------------------------
// phase 2 of the tendency kernel for one line of direction D: Fd = base of the NV tiles holding F^D of this
// element; on return the line holds D_D F^D minus the lifted face terms (eq. 27, 30, 32; App. A3)
// ------------------------------------------------------------------------------------------------
template <int Nq, bool MOIST, bool SGS, int D>
__device__ __forceinline__ void cm5_tend_line(const CmKP& p, double* __restrict__ Fd, const double* __restrict__ Qs,
                                              const double* __restrict__ cs, int l, int e, int4 elz) {
  using C = CmCfg5<Nq, MOIST>;
  constexpr int NP = C::NP, N = Nq - 1, NV = C::NV, NGD = C::NGD, SLOT = C::SLOT, STR = Cm5Str<Nq, D>::value;
  const int erow = elz.y;
  const int nb0 = __ldg(p.nbr + (size_t)e * 6 + 2 * D), nb1 = __ldg(p.nbr + (size_t)e * 6 + 2 * D + 1);
  int base, kline; cm5_line<Nq, D>(l, base, kline);
  const int nlo = base, nhi = base + N * STR;
  // neighbour traces: 6 state values + the SGS values the face-normal flux needs, both ends, issued up front
  double Yp[2][6], gp[2][5];
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    const int nb = s ? nb1 : nb0;
    const size_t idp = (size_t)(nb >= 0 ? nb : e) * NP + (s ? nlo : nhi);     // coincident node on the neighbour's facing plane
#pragma unroll
    for (int v = 0; v < NV; ++v) Yp[s][v] = __ldg(p.Q + v * p.stride + idp);
    if (SGS)
#pragma unroll
      for (int k = 0; k < NGD; ++k) gp[s][k] = __ldg(p.G + (size_t)cm5_gidx(D, k) * p.stride + idp);
  }
  // r = sgn F^D(end) - sJ F*  at the two ends
  double r[2][6];
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    const int nb = s ? nb1 : nb0;
    const int nm = s ? nhi : nlo;
    const double sgn = s ? 1.0 : -1.0;
    const double sJ = p.cA[D], A = sgn * sJ;
    double Ym[6], Ftm[6];
#pragma unroll
    for (int v = 0; v < NV; ++v) { Ym[v] = Qs[v * SLOT + nm]; Ftm[v] = sgn * Fd[v * SLOT + nm]; }
    const double cm_ = cs[nm];
    const double uAm = (Ym[1 + D] * A) * cm_rcp(Ym[0]);                     // sJ (u^- . n)
    CmSite st; CmPrim P;
    if (nb >= 0) {
      cm5_site(p, (D < 2) ? erow + kline : (s ? elz.z : elz.x), st);
      cm_eos<MOIST>(p, Yp[s], st, P);
      double Fp[6];
      cm5_flux_face<MOIST, SGS, D>(Yp[s], P, gp[s], A, Fp);
      const double cp = cm_sqrt(P.c2);
      const double uAp = A * ((D == 0) ? P.u : (D == 1) ? P.v : P.w);
      const double lamsJ = fmax(fabs(uAm) + cm_ * sJ, fabs(uAp) + cp * sJ);  // sJ * lambda (R2)
#pragma unroll
      for (int v = 0; v < NV; ++v) r[s][v] = 0.5 * (Ftm[v] - Fp[v]) - 0.5 * lamsJ * (Ym[v] - Yp[s][v]);
    } else {
      // free-slip wall (A6-A7): Rusanov against the mirrored state = [0; (p' + rho u_n (u_n + lambda)) n; 0; 0];
      // second-order normal fluxes vanish (R10) except the prescribed bottom energy flux
      cm5_site(p, (D < 2) ? erow + kline : (s ? erow + N : erow), st);
      cm_eos<MOIST>(p, Ym, st, P);
      const double un = uAm / sJ;
      const double lam = fabs(un) + cm_;
      const double mom = P.pp + Ym[0] * un * (un + lam);
#pragma unroll
      for (int v = 0; v < NV; ++v) r[s][v] = Ftm[v];
      r[s][1 + D] -= mom * A;
      if (D == 2 && s == 0) r[s][4] += sJ * p.shf;
    }
  }
  // contraction along the line, all variables, lifted face terms folded into the end values
#pragma unroll
  for (int v = 0; v < NV; ++v) {
    double* a = Fd + v * SLOT + base;
    double x[Nq], y[Nq];
#pragma unroll
    for (int m = 0; m < Nq; ++m) x[m] = a[m * STR];
#pragma unroll
    for (int i = 0; i < Nq; ++i) {
      double s = 0.0;
#pragma unroll
      for (int m = 0; m < Nq; ++m) s += p.D[i][m] * x[m];
      y[i] = s;
    }
    y[0] -= p.inv_w0 * r[0][v];
    y[N] -= p.inv_w0 * r[1][v];
#pragma unroll
    for (int i = 0; i < Nq; ++i) a[i * STR] = y[i];
  }
}

template <int Nq, bool MOIST, bool SGS>
__global__ void __launch_bounds__(CmCfg5<Nq, MOIST>::THREADS, CmCfg5<Nq, MOIST>::MINB_T) cm5_tendency_kernel(const __grid_constant__ CmKP p) {
  using C = CmCfg5<Nq, MOIST>;
  constexpr int NF = C::NF, NP = C::NP, NV = C::NV, NG = C::NG, SLOT = C::SLOT, NFP = C::NFP, THREADS = C::THREADS;
  extern __shared__ __align__(128) double smem5[];
  double* Qt = smem5;                                  // [NV][SLOT]   state
  double* Gt = Qt + NV * SLOT;                         // [GS][SLOT]   packed SGS fluxes, then F^1 | F^2
  double* F3t = Gt + C::GS * SLOT;                     // [NV][SLOT]   F^3
  double* ct = F3t + NV * SLOT;                        // [SLOT]       sound speed
  double* Rt = ct + SLOT;                              // [NV][SLOT]   LSRK residual
  uint64_t* mbar = reinterpret_cast<uint64_t*>(Rt + NV * SLOT);   // [2]

  const int t = threadIdx.x;
  const int e = blockIdx.x;
  const bool stagemode = (p.mode != 0);
  const bool readres = stagemode && (p.rka != 0.0);
  const int sh = C::ODD ? (e & 1) : 0;

  if (t == 0) {
    cm5_mbar_init(&mbar[0], 1);
    cm5_mbar_init(&mbar[1], 1);
    cm5_fence_mbar_init();
    const long long src = (long long)e * NP - sh;
    cm5_mbar_expect_tx(&mbar[0], (uint32_t)((NV + (SGS ? NG : 0)) * SLOT * sizeof(double)));
#pragma unroll
    for (int v = 0; v < NV; ++v) cm5_bulk_g2s(Qt + v * SLOT, p.Q + v * p.stride + src, SLOT * 8, &mbar[0]);
    if (SGS)
#pragma unroll
      for (int k = 0; k < NG; ++k) cm5_bulk_g2s(Gt + k * SLOT, p.G + k * p.stride + src, SLOT * 8, &mbar[0]);
    if (readres) {
      cm5_mbar_expect_tx(&mbar[1], (uint32_t)(NV * SLOT * sizeof(double)));
#pragma unroll
      for (int v = 0; v < NV; ++v) cm5_bulk_g2s(Rt + v * SLOT, p.dQ + v * p.stride + src, SLOT * 8, &mbar[1]);
    }
  }
  const int4 elz = __ldg(reinterpret_cast<const int4*>(p.elz) + e);
  double* Qs = Qt + sh; double* Gs = Gt + sh; double* F3 = F3t + sh; double* cs = ct + sh; const double* Rs = Rt + sh;
  const int n = t;
  const bool node = t < NP;
  CmSite st;
  if (node) cm5_site(p, elz.y + n / NF, st);
  __syncthreads();                                     // mbarrier init visible to the waiters
  cm5_mbar_wait(&mbar[0], 0);

  // ---- phase 1: primitives and contravariant fluxes of the own node (F^1, F^2 overwrite the G slots in place)
  double buoy = 0.0;
  if (node) {
    double Y[6], g[12]; CmPrim P;
#pragma unroll
    for (int v = 0; v < NV; ++v) Y[v] = Qs[v * SLOT + n];
    if (SGS)
#pragma unroll
      for (int k = 0; k < NG; ++k) g[k] = Gs[k * SLOT + n];
    cm_eos<MOIST>(p, Y, st, P);
    buoy = P.drho * p.th.grav;
    cs[n] = cm_sqrt(P.c2);
    double Fa[6];
    cm_flux_axis<MOIST, 0>(Y, P, SGS, g, p.cA[0], Fa);
#pragma unroll
    for (int v = 0; v < NV; ++v) Gs[v * SLOT + n] = Fa[v];
    cm_flux_axis<MOIST, 1>(Y, P, SGS, g, p.cA[1], Fa);
#pragma unroll
    for (int v = 0; v < NV; ++v) Gs[(NV + v) * SLOT + n] = Fa[v];
    cm_flux_axis<MOIST, 2>(Y, P, SGS, g, p.cA[2], Fa);
#pragma unroll
    for (int v = 0; v < NV; ++v) F3[v * SLOT + n] = Fa[v];
  }
  __syncthreads();

  // ---- phase 2: one thread per line, one (set of) warp(s) per direction
  for (int lt = t; lt < 3 * NFP; lt += THREADS) {
    const int d = lt / NFP, l = lt % NFP;
    if (l < NF) {
      if (d == 0) cm5_tend_line<Nq, MOIST, SGS, 0>(p, Gs, Qs, cs, l, e, elz);
      else if (d == 1) cm5_tend_line<Nq, MOIST, SGS, 1>(p, Gs + NV * SLOT, Qs, cs, l, e, elz);
      else cm5_tend_line<Nq, MOIST, SGS, 2>(p, F3, Qs, cs, l, e, elz);
    }
  }
  __syncthreads();

  // ---- phase 3: assemble the tendency of the own node and update
  if (node) {
    if (readres) cm5_mbar_wait(&mbar[1], 0);
    const size_t idx = (size_t)e * NP + n;
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      const double a = Gs[v * SLOT + n] + Gs[(NV + v) * SLOT + n] + F3[v * SLOT + n];
      double rhs = -p.invJ * a;
      if (v == 3) rhs -= buoy;                                   // -(rho - rho_r) grad Phi   (eq. 4)
      if (!stagemode) {
        __stcs(p.dQ + v * p.stride + idx, rhs);
      } else {
        // a5: dU <- A_s dU + dt RHS ; U <- U + B_s dU
        const double dold = readres ? Rs[v * SLOT + n] : 0.0;
        const double dnew = p.rka * dold + p.dt * rhs;
        __stcs(p.dQ + v * p.stride + idx, dnew);
        __stcs(p.Qnew + v * p.stride + idx, Qs[v * SLOT + n] + p.rkb * dnew);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// a2: auxiliary gradient + Smagorinsky-Lilly (flat bricks), same decomposition
// ------------------------------------------------------------------------------------------------
template <int Nq, bool MOIST, int D>
__device__ __forceinline__ void cm5_grad_line(const CmKP& p, const double* __restrict__ ss, double* __restrict__ dd, int l, int e, int4 elz) {
  using C = CmCfg5<Nq, MOIST>;
  constexpr int NP = C::NP, N = Nq - 1, NV = C::NV, NS = C::NS, SLOT = C::SLOT, STR = Cm5Str<Nq, D>::value;
  const int erow = elz.y;
  const int nb0 = __ldg(p.nbr + (size_t)e * 6 + 2 * D), nb1 = __ldg(p.nbr + (size_t)e * 6 + 2 * D + 1);
  int base, kline; cm5_line<Nq, D>(l, base, kline);
  const int nlo = base, nhi = base + N * STR;
  double Yp[2][6];
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    const int nb = s ? nb1 : nb0;
    const size_t idp = (size_t)(nb >= 0 ? nb : e) * NP + (s ? nlo : nhi);
#pragma unroll
    for (int v = 0; v < NV; ++v) Yp[s][v] = __ldg(p.Q + v * p.stride + idp);
  }
  double dl[2][5];                                      // s* - s^- at the two ends (eq. 30-31: central flux)
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    const int nb = s ? nb1 : nb0;
    const int nm = s ? nhi : nlo;
    if (nb >= 0) {
      const int row = (D < 2) ? erow + kline : (s ? elz.z : elz.x);
      double sp[5];
      cm5_eos_grad<MOIST>(p, Yp[s], __ldg(p.ztab + (size_t)row * CM_ZTAB_W), sp);
#pragma unroll
      for (int v = 0; v < NS; ++v) dl[s][v] = 0.5 * (sp[v] - ss[v * SLOT + nm]);
    } else {
      // wall: u_bc = u^- - (n.u^-) n  (A6); scalars unchanged (A8)
#pragma unroll
      for (int v = 0; v < NS; ++v) dl[s][v] = (v == D) ? -ss[v * SLOT + nm] : 0.0;
    }
  }
#pragma unroll
  for (int v = 0; v < NS; ++v) {
    const double* in = ss + v * SLOT + base;
    double* out = dd + v * SLOT + base;
    double x[Nq];
#pragma unroll
    for (int m = 0; m < Nq; ++m) x[m] = in[m * STR];
#pragma unroll
    for (int i = 0; i < Nq; ++i) {
      double a = 0.0;
#pragma unroll
      for (int m = 0; m < Nq; ++m) a += p.D[i][m] * x[m];
      if (i == 0) a -= p.inv_w0 * dl[0][v];
      if (i == N) a += p.inv_w0 * dl[1][v];
      out[i * STR] = a;
    }
  }
}

template <int Nq, bool MOIST>
__global__ void __launch_bounds__(CmCfg5<Nq, MOIST>::THREADS, CmCfg5<Nq, MOIST>::MINB_G) cm5_gradient_kernel(const __grid_constant__ CmKP p) {
  using C = CmCfg5<Nq, MOIST>;
  constexpr int NF = C::NF, NP = C::NP, NV = C::NV, NS = C::NS, SLOT = C::SLOT, NFP = C::NFP, THREADS = C::THREADS;
  extern __shared__ __align__(128) double smem5[];
  double* Qt = smem5;                                  // [NV][SLOT]      state, then the gradient variables in place
  double* dt_ = Qt + NV * SLOT;                        // [3][NS][SLOT]   reference-space derivatives + lifted jumps
  uint64_t* mbar = reinterpret_cast<uint64_t*>(dt_ + 3 * NS * SLOT);

  const int t = threadIdx.x;
  const int e = blockIdx.x;
  const int sh = C::ODD ? (e & 1) : 0;
  if (t == 0) {
    cm5_mbar_init(&mbar[0], 1);
    cm5_fence_mbar_init();
    const long long src = (long long)e * NP - sh;
    cm5_mbar_expect_tx(&mbar[0], (uint32_t)(NV * SLOT * sizeof(double)));
#pragma unroll
    for (int v = 0; v < NV; ++v) cm5_bulk_g2s(Qt + v * SLOT, p.Q + v * p.stride + src, SLOT * 8, &mbar[0]);
  }
  const int4 elz = __ldg(reinterpret_cast<const int4*>(p.elz) + e);
  double* ss = Qt + sh; double* dd = dt_ + sh;
  const int n = t;
  const bool node = t < NP;
  double Phi = 0.0;
  if (node) Phi = __ldg(p.ztab + (size_t)(elz.y + n / NF) * CM_ZTAB_W);
  __syncthreads();
  cm5_mbar_wait(&mbar[0], 0);

  // ---- phase 1: gradient variables of the own node, in place of the state
  if (node) {
    double Y[6], s[5];
#pragma unroll
    for (int v = 0; v < NV; ++v) Y[v] = ss[v * SLOT + n];
    cm5_eos_grad<MOIST>(p, Y, Phi, s);
#pragma unroll
    for (int v = 0; v < NS; ++v) ss[v * SLOT + n] = s[v];
  }
  __syncthreads();

  // ---- phase 2: one thread per line
  for (int lt = t; lt < 3 * NFP; lt += THREADS) {
    const int d = lt / NFP, l = lt % NFP;
    if (l < NF) {
      if (d == 0) cm5_grad_line<Nq, MOIST, 0>(p, ss, dd, l, e, elz);
      else if (d == 1) cm5_grad_line<Nq, MOIST, 1>(p, ss, dd + NS * SLOT, l, e, elz);
      else cm5_grad_line<Nq, MOIST, 2>(p, ss, dd + 2 * NS * SLOT, l, e, elz);
    }
  }
  __syncthreads();

  // ---- phase 3: physical gradient, closure, store
  if (node) {
    const size_t idx = (size_t)e * NP + n;
    double Gr[5][3];
#pragma unroll
    for (int v = 0; v < NS; ++v)
#pragma unroll
      for (int c = 0; c < 3; ++c) Gr[v][c] = (p.cA[c] * p.invJ) * dd[(c * NS + v) * SLOT + n];
    if (!MOIST) { Gr[4][0] = Gr[4][1] = Gr[4][2] = 0.0; }
    if (p.mode == 1) {
#pragma unroll
      for (int v = 0; v < 5; ++v)
#pragma unroll
        for (int c = 0; c < 3; ++c) __stcs(p.Gout + (size_t)(3 * v + c) * p.stride + idx, Gr[v][c]);
    } else {
      // eq. (33)-(38): S, nu_t = (C_s Delta)^2 sqrt(2 S:S), D_t = nu_t / Pr_t; store tau, J + D, d_q
      const double Sxx = Gr[0][0], Syy = Gr[1][1], Szz = Gr[2][2];
      const double Sxy = 0.5 * (Gr[0][1] + Gr[1][0]), Sxz = 0.5 * (Gr[0][2] + Gr[2][0]), Syz = 0.5 * (Gr[1][2] + Gr[2][1]);
      const double ss2 = Sxx * Sxx + Syy * Syy + Szz * Szz + 2.0 * (Sxy * Sxy + Sxz * Sxz + Syz * Syz);
      const double nu = p.cs2delta2 * cm_sqrt(2.0 * ss2);
      const double m2nu = -2.0 * nu, mDt = -nu * p.inv_Pr;
      double* o = p.Gout + idx;
      const long long st = p.stride;
      o[0] = m2nu * Sxx; o[st] = m2nu * Syy; o[2 * st] = m2nu * Szz;
      o[3 * st] = m2nu * Sxy; o[4 * st] = m2nu * Sxz; o[5 * st] = m2nu * Syz;
      o[6 * st] = mDt * Gr[3][0]; o[7 * st] = mDt * Gr[3][1]; o[8 * st] = mDt * Gr[3][2];
      if (MOIST) { o[9 * st] = mDt * Gr[4][0]; o[10 * st] = mDt * Gr[4][1]; o[11 * st] = mDt * Gr[4][2]; }
    }
  }
}
