// cm_dg_kernels4.cuh -- the hot kernels for flat bricks (GEOM == 0): ONE WARP PER ELEMENT, no CTA barriers.
//
// Why: the thread-per-node kernels (cm_dg_kernels2.cuh) spend 1500 warp instructions per node-thread, 600 M shared
// memory wavefronts per launch and three CTA barriers per element batch; ncu shows them bound by the L1/shared
// pipe (61 %) and by latency (0.48 eligible warps per scheduler), not by DRAM (31 %) -- profiles/r1a_v2.md.  Here
//   * a warp owns an element from load to store; the only synchronisation is __syncwarp(), so the 9 warps of an SM
//     drift apart and overlap each other's load, flux, contraction and store phases on their own;
//   * phase 1 and 3 are FLAT: lane l owns nodes l, l+32, l+64, ... (coalesced 256-byte LDG / STG rows straight
//     from / to the structure-of-arrays state; NPL independent nodes per lane = instruction-level parallelism);
//   * phase 2 is one LINE ROUND per direction: lane l owns line l of that direction (25 of 32 lanes at N = 4),
//     pulls its Nq values per variable from shared memory, applies D (constant-bank operands) in registers, and
//     ALSO evaluates the numerical flux at the line's two end nodes (Rusanov + central SGS flux against the
//     neighbour's trace, or the wall rule) and folds the lifted result into the two end values before writing the
//     line back in place.  No face buffers, no second pass over the face nodes, and every shared-memory operand is
//     touched 4 times per (variable, direction): flux store, line load, line store, assembly load;
//   * nothing but the contravariant fluxes (3 NV tiles), the state (NV tiles) and the sound speed (1 tile) lives
//     in shared memory: 25 KB per warp at N = 4 with moisture -> 3 CTAs x 3 warps per SM.
// Arithmetic follows cm_dg_physics.cuh (R12 pressure perturbation, MUFU-seeded rcp / sqrt).  P:L<n> = paper line.
#pragma once
#include "cm_dg_internal.h"
#include "cm_dg_physics.cuh"

template <int Nq, bool MOIST> struct CmCfg4 {
  static constexpr int NF = Nq * Nq;
  static constexpr int NP = Nq * Nq * Nq;
  static constexpr int NV = MOIST ? 6 : 5;
  static constexpr int NG = MOIST ? 12 : 9;
  static constexpr int NS = MOIST ? 5 : 4;                  // gradient variables u, v, w, h_tot, [q]
  static constexpr int NGD = MOIST ? 5 : 4;                 // SGS values one face direction needs
  static constexpr int NPL = (NP + 31) / 32;                // nodes per lane (flat phases)
  static constexpr int LR = (NF + 31) / 32;                 // sub-rounds of a line round
  static constexpr int TEND_D = (3 * NV + NV + 1) * NP;     // doubles per warp: F[3][NV], Q[NV], c
  static constexpr int GRAD_D = (NS + 3 * NS) * NP;         // doubles per warp: s[NS], ds/dxi_d [3][NS]
  // warps per CTA / CTAs per SM that maximise resident warps within 228 KB (1 KB reserved per CTA)
  static constexpr int ctas(int w, int doubles) { return (int)(233472 / (w * doubles * 8 + 1024)); }
  static constexpr int cap(int v, int hi) { return v > hi ? hi : v; }
  static constexpr int best_w(int doubles) {
    int bw = 1, best = 0;
    for (int w = 1; w <= 4; ++w) { const int n = cap(w * cap(ctas(w, doubles), 32), 16); if (n >= best && ctas(w, doubles) >= 1) { best = n; bw = w; } }
    return bw;
  }
  static constexpr int WT = best_w(TEND_D), WG = best_w(GRAD_D);
  static constexpr int MINB_T = cap(ctas(WT, TEND_D), 16 / WT) < 1 ? 1 : cap(ctas(WT, TEND_D), 16 / WT);
  static constexpr int MINB_G = cap(ctas(WG, GRAD_D), 16 / WG) < 1 ? 1 : cap(ctas(WG, GRAD_D), 16 / WG);
  static constexpr size_t TEND_SMEM = sizeof(double) * WT * TEND_D;
  static constexpr size_t GRAD_SMEM = sizeof(double) * WG * GRAD_D;
};

__device__ __forceinline__ void cm4_site(const CmKP& p, int row, CmSite& s) {
  const double2* t = reinterpret_cast<const double2*>(p.ztab + (size_t)row * CM_ZTAB_W);
  const double2 a = __ldg(t), b = __ldg(t + 1), c = __ldg(t + 2), d = __ldg(t + 3);
  s.Phi = a.x; s.rho_r = a.y; s.rhoe_r = b.x; s.rhoq_r = b.y; s.E_r = c.x; s.q_r = c.y; s.icvm_r = d.x;
}

// primitives the gradient needs (u, v, w, h_tot, q): eq. (6)-(10), (13)-(14)
template <bool MOIST>
__device__ __forceinline__ void cm4_eos_grad(const CmKP& p, const double* Y, double Phi, double* s) {
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
__host__ __device__ constexpr int cm4_gidx(int d, int k) {
  return (k == 3) ? 6 + d : (k == 4) ? 9 + d : (k == d) ? d : k + d + 2;   // (0,1)->3, (0,2)->4, (1,2)->5
}

// contravariant flux along axis D, A = s * e_D; gd = the SGS values that axis needs: tau(D,0..2), (J+D)_D, [d_q,D]
template <bool MOIST, bool SGS, int D>
__device__ __forceinline__ void cm4_flux_face(const double* Y, const CmPrim& P, const double* gd, double s, double* Fn) {
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

// geometry of line l of direction D: first node, node stride, zeta index of the line (D < 2)
template <int Nq, int D>
__device__ __forceinline__ void cm4_line(int l, int& base, int& kline) {
  constexpr int NF = Nq * Nq;
  const int a = l % Nq, b = l / Nq;
  base = (D == 0) ? Nq * l : (D == 1) ? a + NF * b : l;
  kline = b;
}
template <int Nq, int D> struct Cm4Str { static constexpr int value = (D == 0) ? 1 : (D == 1) ? Nq : Nq * Nq; };

// ------------------------------------------------------------------------------------------------
// a3-a5: one line round of the tendency kernel: D_d F^d along every line of direction D, in place, with the
// lifted numerical flux of the two faces normal to D folded into the end nodes (eq. 27, 30, 32; App. A3)
// ------------------------------------------------------------------------------------------------
template <int Nq, bool MOIST, bool SGS, int D>
__device__ __forceinline__ void cm4_tend_round(const CmKP& p, double* __restrict__ Fd, const double* __restrict__ Qs,
                                               const double* __restrict__ cs, int lane, int e, int erow, int4 elz) {
  using C = CmCfg4<Nq, MOIST>;
  constexpr int NF = C::NF, NP = C::NP, N = Nq - 1, NV = C::NV, NGD = C::NGD, STR = Cm4Str<Nq, D>::value;
  const int nb0 = __ldg(p.nbr + (size_t)e * 6 + 2 * D), nb1 = __ldg(p.nbr + (size_t)e * 6 + 2 * D + 1);
#pragma unroll
  for (int sub = 0; sub < C::LR; ++sub) {
    const int l = lane + 32 * sub;
    if (l < NF) {
      int base, kline; cm4_line<Nq, D>(l, base, kline);
      const int nlo = base, nhi = base + N * STR;
      // neighbour traces: 6 state values + the SGS values the face-normal flux needs, both ends, issued up front
      double Yp[2][6], gp[2][5];
#pragma unroll
      for (int s = 0; s < 2; ++s) {
        const int nb = s ? nb1 : nb0;
        if (nb >= 0) {
          const size_t idp = (size_t)nb * NP + (s ? nlo : nhi);     // coincident node on the neighbour's facing plane
#pragma unroll
          for (int v = 0; v < NV; ++v) Yp[s][v] = __ldg(p.Q + v * p.stride + idp);
          if (SGS)
#pragma unroll
            for (int k = 0; k < NGD; ++k) gp[s][k] = __ldg(p.G + (size_t)cm4_gidx(D, k) * p.stride + idp);
        }
      }
      double B[2][6], alpha[2];
#pragma unroll
      for (int s = 0; s < 2; ++s) {
        const int nb = s ? nb1 : nb0;
        const int nm = s ? nhi : nlo;
        const double sgn = s ? 1.0 : -1.0;
        const double sJ = p.cA[D], A = sgn * sJ;
        double Ym[6];
#pragma unroll
        for (int v = 0; v < NV; ++v) Ym[v] = Qs[v * NP + nm];
        const double cm_ = cs[nm];
        const double uAm = (Ym[1 + D] * A) * cm_rcp(Ym[0]);                     // sJ (u^- . n)
        CmSite st; CmPrim P;
        if (nb >= 0) {
          cm4_site(p, (D < 2) ? erow + kline : (s ? elz.z : elz.x), st);
          cm_eos<MOIST>(p, Yp[s], st, P);
          double Fp[6];
          cm4_flux_face<MOIST, SGS, D>(Yp[s], P, gp[s], A, Fp);
          const double cp = cm_sqrt(P.c2);
          const double uAp = A * ((D == 0) ? P.u : (D == 1) ? P.v : P.w);
          const double lamsJ = fmax(fabs(uAm) + cm_ * sJ, fabs(uAp) + cp * sJ);  // sJ * lambda (R2)
#pragma unroll
          for (int v = 0; v < NV; ++v) B[s][v] = 0.5 * Fp[v] + 0.5 * lamsJ * (Ym[v] - Yp[s][v]);
          alpha[s] = 0.5 * sgn;
        } else {
          // free-slip wall (A6-A7): Rusanov against the mirrored state = [0; (p' + rho u_n (u_n + lambda)) n; 0; 0];
          // second-order normal fluxes vanish (R10) except the prescribed bottom energy flux
          cm4_site(p, (D < 2) ? erow + kline : (s ? erow + N : erow), st);
          cm_eos<MOIST>(p, Ym, st, P);
          const double un = uAm / sJ;
          const double lam = fabs(un) + cm_;
          const double mom = P.pp + Ym[0] * un * (un + lam);
#pragma unroll
          for (int v = 0; v < NV; ++v) B[s][v] = 0.0;
          B[s][1 + D] = mom * A;
          if (D == 2 && s == 0) B[s][4] = -sJ * p.shf;
          alpha[s] = sgn;
        }
      }
      // contraction along the line, all variables; r = alpha F^d(end) - B is the lifted face term
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        double* a = Fd + v * NP + base;
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
        y[0] -= p.inv_w0 * (alpha[0] * x[0] - B[0][v]);
        y[N] -= p.inv_w0 * (alpha[1] * x[N] - B[1][v]);
#pragma unroll
        for (int i = 0; i < Nq; ++i) a[i * STR] = y[i];
      }
    }
  }
}

template <int Nq, bool MOIST, bool SGS>
__global__ void __launch_bounds__(32 * CmCfg4<Nq, MOIST>::WT, 1) cm4_tendency_kernel(const __grid_constant__ CmKP p) {
  using C = CmCfg4<Nq, MOIST>;
  constexpr int NF = C::NF, NP = C::NP, NV = C::NV, NG = C::NG, NPL = C::NPL;
  extern __shared__ __align__(16) double smem4[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  double* F = smem4 + (size_t)warp * C::TEND_D;        // [3][NV][NP]  contravariant fluxes, then D_d F^d - lift
  double* Qs = F + 3 * NV * NP;                        // [NV][NP]     state
  double* cs = Qs + NV * NP;                           // [NP]         sound speed
  const bool stagemode = (p.mode != 0);
  const bool readres = stagemode && (p.rka != 0.0);
  const int e_first = ((int)blockIdx.x * C::WT + warp) * p.epw;

  for (int r = 0; r < p.epw; ++r) {
    const int e = e_first + r;
    if (e >= p.Ne) break;
    const int4 elz = __ldg(reinterpret_cast<const int4*>(p.elz) + e);
    const int erow = elz.y;

    // ---- phase 1 (flat): primitives and contravariant fluxes of the own nodes -> shared memory
    double buoy[NPL];
#pragma unroll
    for (int m = 0; m < NPL; ++m) {
      const int n = lane + 32 * m;
      buoy[m] = 0.0;
      if (n < NP) {
        const size_t idx = (size_t)e * NP + n;
        double Y[6], g[12]; CmSite st; CmPrim P;
        cm_load_state<NV>(p.Q, p.stride, idx, Y);
        if (SGS) cm_load_state<NG>(p.G, p.stride, idx, g);
        cm4_site(p, erow + n / NF, st);
        cm_eos<MOIST>(p, Y, st, P);
        buoy[m] = P.drho * p.th.grav;
        cs[n] = cm_sqrt(P.c2);
#pragma unroll
        for (int v = 0; v < NV; ++v) Qs[v * NP + n] = Y[v];
        double Fa[6];
        cm_flux_axis<MOIST, 0>(Y, P, SGS, g, p.cA[0], Fa);
#pragma unroll
        for (int v = 0; v < NV; ++v) F[v * NP + n] = Fa[v];
        cm_flux_axis<MOIST, 1>(Y, P, SGS, g, p.cA[1], Fa);
#pragma unroll
        for (int v = 0; v < NV; ++v) F[(NV + v) * NP + n] = Fa[v];
        cm_flux_axis<MOIST, 2>(Y, P, SGS, g, p.cA[2], Fa);
#pragma unroll
        for (int v = 0; v < NV; ++v) F[(2 * NV + v) * NP + n] = Fa[v];
      }
    }
    // the residual is fetched while the line rounds run (streaming: keep L2 for the Q / G traces)
    double dold[NPL][NV];
#pragma unroll
    for (int m = 0; m < NPL; ++m) {
      const int n = lane + 32 * m;
#pragma unroll
      for (int v = 0; v < NV; ++v) dold[m][v] = (readres && n < NP) ? __ldcs(p.dQ + v * p.stride + (size_t)e * NP + n) : 0.0;
    }
    __syncwarp();

    // ---- phase 2: line rounds (contraction + both end faces) along xi, eta, zeta
    cm4_tend_round<Nq, MOIST, SGS, 0>(p, F, Qs, cs, lane, e, erow, elz);
    cm4_tend_round<Nq, MOIST, SGS, 1>(p, F + NV * NP, Qs, cs, lane, e, erow, elz);
    cm4_tend_round<Nq, MOIST, SGS, 2>(p, F + 2 * NV * NP, Qs, cs, lane, e, erow, elz);
    __syncwarp();

    // ---- phase 3 (flat): assemble the tendency of the own nodes and update
#pragma unroll
    for (int m = 0; m < NPL; ++m) {
      const int n = lane + 32 * m;
      if (n < NP) {
        const size_t idx = (size_t)e * NP + n;
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          const double a = F[v * NP + n] + F[(NV + v) * NP + n] + F[(2 * NV + v) * NP + n];
          double rhs = -p.invJ * a;
          if (v == 3) rhs -= buoy[m];                                // -(rho - rho_r) grad Phi   (eq. 4)
          if (!stagemode) {
            __stcs(p.dQ + v * p.stride + idx, rhs);
          } else {
            // a5: dU <- A_s dU + dt RHS ; U <- U + B_s dU
            const double dnew = p.rka * dold[m][v] + p.dt * rhs;
            __stcs(p.dQ + v * p.stride + idx, dnew);
            __stcs(p.Qnew + v * p.stride + idx, Qs[v * NP + n] + p.rkb * dnew);
          }
        }
      }
    }
    __syncwarp();
  }
}

// ------------------------------------------------------------------------------------------------
// a2: auxiliary gradient + Smagorinsky-Lilly (flat bricks), same decomposition
// ------------------------------------------------------------------------------------------------
template <int Nq, bool MOIST, int D>
__device__ __forceinline__ void cm4_grad_round(const CmKP& p, const double* __restrict__ s_sh, double* __restrict__ dd, int lane,
                                               int e, int erow, int4 elz) {
  using C = CmCfg4<Nq, MOIST>;
  constexpr int NF = C::NF, NP = C::NP, N = Nq - 1, NV = C::NV, NS = C::NS, STR = Cm4Str<Nq, D>::value;
  const int nb0 = __ldg(p.nbr + (size_t)e * 6 + 2 * D), nb1 = __ldg(p.nbr + (size_t)e * 6 + 2 * D + 1);
#pragma unroll
  for (int sub = 0; sub < C::LR; ++sub) {
    const int l = lane + 32 * sub;
    if (l < NF) {
      int base, kline; cm4_line<Nq, D>(l, base, kline);
      const int nlo = base, nhi = base + N * STR;
      double Yp[2][6];
#pragma unroll
      for (int s = 0; s < 2; ++s) {
        const int nb = s ? nb1 : nb0;
        if (nb >= 0) {
          const size_t idp = (size_t)nb * NP + (s ? nlo : nhi);
#pragma unroll
          for (int v = 0; v < NV; ++v) Yp[s][v] = __ldg(p.Q + v * p.stride + idp);
        }
      }
      double dl[2][5];                                  // s* - s^- at the two ends (eq. 30-31: central flux)
#pragma unroll
      for (int s = 0; s < 2; ++s) {
        const int nb = s ? nb1 : nb0;
        const int nm = s ? nhi : nlo;
        if (nb >= 0) {
          const int row = (D < 2) ? erow + kline : (s ? elz.z : elz.x);
          double sp[5];
          cm4_eos_grad<MOIST>(p, Yp[s], __ldg(p.ztab + (size_t)row * CM_ZTAB_W), sp);
#pragma unroll
          for (int v = 0; v < NS; ++v) dl[s][v] = 0.5 * (sp[v] - s_sh[v * NP + nm]);
        } else {
          // wall: u_bc = u^- - (n.u^-) n  (A6); scalars unchanged (A8)
#pragma unroll
          for (int v = 0; v < NS; ++v) dl[s][v] = (v == D) ? -s_sh[v * NP + nm] : 0.0;
        }
      }
#pragma unroll
      for (int v = 0; v < NS; ++v) {
        const double* in = s_sh + v * NP + base;
        double* out = dd + v * NP + base;
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
  }
}

template <int Nq, bool MOIST>
__global__ void __launch_bounds__(32 * CmCfg4<Nq, MOIST>::WG, CmCfg4<Nq, MOIST>::MINB_G) cm4_gradient_kernel(const __grid_constant__ CmKP p) {
  using C = CmCfg4<Nq, MOIST>;
  constexpr int NF = C::NF, NP = C::NP, NV = C::NV, NS = C::NS, NPL = C::NPL;
  extern __shared__ __align__(16) double smem4[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  double* s_sh = smem4 + (size_t)warp * C::GRAD_D;     // [NS][NP]      gradient variables
  double* d_sh = s_sh + NS * NP;                       // [3][NS][NP]   reference-space derivatives + lifted jumps
  const int e_first = ((int)blockIdx.x * C::WG + warp) * p.epw;

  for (int r = 0; r < p.epw; ++r) {
    const int e = e_first + r;
    if (e >= p.Ne) break;
    const int4 elz = __ldg(reinterpret_cast<const int4*>(p.elz) + e);
    const int erow = elz.y;

    // ---- phase 1 (flat): gradient variables of the own nodes
#pragma unroll
    for (int m = 0; m < NPL; ++m) {
      const int n = lane + 32 * m;
      if (n < NP) {
        double Y[6], s[5];
        cm_load_state<NV>(p.Q, p.stride, (size_t)e * NP + n, Y);
        cm4_eos_grad<MOIST>(p, Y, __ldg(p.ztab + (size_t)(erow + n / NF) * CM_ZTAB_W), s);
#pragma unroll
        for (int v = 0; v < NS; ++v) s_sh[v * NP + n] = s[v];
      }
    }
    __syncwarp();

    // ---- phase 2: line rounds
    cm4_grad_round<Nq, MOIST, 0>(p, s_sh, d_sh, lane, e, erow, elz);
    cm4_grad_round<Nq, MOIST, 1>(p, s_sh, d_sh + NS * NP, lane, e, erow, elz);
    cm4_grad_round<Nq, MOIST, 2>(p, s_sh, d_sh + 2 * NS * NP, lane, e, erow, elz);
    __syncwarp();

    // ---- phase 3 (flat): physical gradient, closure, store
#pragma unroll
    for (int m = 0; m < NPL; ++m) {
      const int n = lane + 32 * m;
      if (n < NP) {
        const size_t idx = (size_t)e * NP + n;
        double Gr[5][3];
#pragma unroll
        for (int v = 0; v < NS; ++v)
#pragma unroll
          for (int c = 0; c < 3; ++c) Gr[v][c] = (p.cA[c] * p.invJ) * d_sh[(c * NS + v) * NP + n];
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
          const double ss = Sxx * Sxx + Syy * Syy + Szz * Szz + 2.0 * (Sxy * Sxy + Sxz * Sxz + Syz * Syz);
          const double nu = p.cs2delta2 * cm_sqrt(2.0 * ss);
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
    __syncwarp();
  }
}
