// cm_dg_kernels7.cuh -- the hot kernels for flat bricks (GEOM == 0): one small CTA per element, every input staged
// asynchronously at CTA start, face work and line work decoupled so that all warps stay busy.
//
// Lessons built in (profiles/r1c_v5.md, profiles/r1e_v9.md, profiles/r1f_prefetch.md): at ~20 resident warps per SM (shared memory holds five
// elements per SM) the kernels are bound by the dependent instruction chain of each warp and by the shared-memory
// data pipe, so no warp may idle at a barrier and nothing may wait on a chain of global loads:
//   * the launch grid IS the tiled element order: element position, neighbour ids, wall flags and z rows follow from
//     blockIdx by integer arithmetic, no connectivity array is read;
//   * tendency kernel (cm7_tendency_kernel):
//       - CTA start: lane 0 of the last warp fetches the element's own Q, packed SGS fluxes G and LSRK residual by 1-D
//         bulk TMA (cp.async.bulk ... mbarrier::complete_tx); every thread copies the neighbour traces of one or two
//         face nodes (6 state values + the 5 SGS values the face-normal flux needs) and the z-table rows with 8-byte
//         cp.async;
//       - phase 1 (thread per node) needs only the TMA data: EOS + contravariant fluxes F^1, F^3 (in place of G) and
//         F^2 (own tiles with a padded zeta-plane stride, so that no line direction has bank conflicts); the cp.async
//         traces land meanwhile;
//       - phase 2, no barrier inside: FACE tasks (thread per face node, direction-generic code, handed out from the
//         last thread downwards so the warp without line tasks takes the second round) turn the trace into the lifted
//         numerical-flux part  rf = -(1/2) sJ n.F^+ - (1/2) sJ lambda (Y^- - Y^+)  in place of the trace, and LINE
//         tasks (thread per line, one warp per direction, D from the constant bank) contract D_d F^d in place, folding
//         the element's own half (1/2) sJ n.F^- of the face term into the line's end values from registers -- the two
//         kinds of task touch disjoint data;
//       - phase 3 (thread per node): all shared-memory operands loaded up front, sum of the three directions, the rf of
//         the up to three faces the node lies on, gravity source, fused LSRK update, coalesced streaming stores;
//       three CTA barriers, 45.5 KB of shared memory and 92 registers per thread at N = 4 moist: five CTAs per SM;
//   * both kernels: the lanes next to the one that issues the bulk copies prefetch the tiles of the element one wave of
//     resident CTAs further on in the launch order into L2 (cp.async.bulk.prefetch.L2), so that bulk copies and trace
//     gathers hit L2 instead of waiting on DRAM (CmKP::ahead);
//   * gradient kernel (cm9_gradient_kernel, at the end of this file): its phases are short enough that the line task
//     can own the face terms of its two end nodes; the 2 x 6 trace values are loaded into REGISTERS at CTA start (in
//     flight together with the TMA) and consumed in phase 2: no trace buffer at all.  cm7_gradient_kernel (trace
//     buffer, as the tendency kernel) remains for the orders whose CTAs have fewer threads than line tasks (N <= 3).
// Arithmetic follows cm_dg_physics.cuh.  P:L<n> = paper line.
#pragma once
#include "cm_dg_internal.h"
#include "cm_dg_physics.cuh"

// ------------------------------------------------------------------------------------------------ PTX helpers
__device__ __forceinline__ uint32_t cm7_saddr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cm7_mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(cm7_saddr(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void cm7_mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(cm7_saddr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cm7_mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "LAB_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra LAB_WAIT;\n"
      "DONE:\n"
      "}\n" ::"r"(cm7_saddr(bar)), "r"(parity) : "memory");
}
// 1-D bulk TMA global -> shared, completion counted in bytes on an mbarrier (16-byte aligned src, dst, size)
__device__ __forceinline__ void cm7_bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(cm7_saddr(dst)),
               "l"(src), "r"(bytes), "r"(cm7_saddr(bar)) : "memory");
}
// L2 prefetch of a contiguous range (16-byte aligned address and size): no destination, no completion to wait for
__device__ __forceinline__ void cm7_prefetch_l2(const void* src, uint32_t bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}
// same with the shared-memory addresses already converted (issue loops: one add per operand and copy)
__device__ __forceinline__ void cm7_bulk_g2s_raw(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src),
               "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void cm7_fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void cm7_cp8(void* dst, const void* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(cm7_saddr(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cm7_cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cm7_cp_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void cm7_cp_wait_but_one() { asm volatile("cp.async.wait_group 1;" ::: "memory"); }

#ifndef CM_LINE_UNROLL
#define CM_LINE_UNROLL 3   // variables per unrolled body of the tendency line task (code size vs ILP: profiles/r2_rowsweep.md)
#endif
#define CM_ZSM_W 10   // doubles per z-table row in shared memory (CmCfg7::ZW)

template <int Nq, bool MOIST> struct CmCfg7 {
  static constexpr int NF = Nq * Nq;
  static constexpr int NP = Nq * Nq * Nq;
  static constexpr int NV = MOIST ? 6 : 5;
  static constexpr int NG = MOIST ? 12 : 9;
  static constexpr int NS = MOIST ? 5 : 4;                  // gradient variables u, v, w, h_tot, [q]
  static constexpr int NGD = MOIST ? 5 : 4;                 // SGS values one face direction needs
  static constexpr int NTR = NV + NGD;                      // trace values per face node (tendency)
  static constexpr int ODD = NP & 1;
  static constexpr int SLOT = NP + ODD;                     // doubles per field tile in shared memory (16-byte multiple)
  static constexpr int THREADS = ((NP + 31) / 32) * 32;
  static constexpr int NFP = ((NF + 31) / 32) * 32;         // line tasks of one direction, padded to whole warps
  static constexpr int ZR = Nq + 2;                         // z-table rows: facing row below, own Nq rows, facing row above
  static constexpr int ZW = 10;                             // doubles per z row in shared memory: rows fall into disjoint banks
  static constexpr int TAIL = (ZR - 1) * ZW + 7 + 1;        // z rows (7 values used per row), mbarrier
  // stride between the trace blocks of two faces: >= rows * NF and = NF (mod 16), so that consecutive face nodes of a
  // warp that straddles two faces fall into consecutive banks
  static constexpr int fstride(int rows) { return rows * NF + ((NF - rows * NF) % 16 + 16) % 16; }
  static constexpr int TS_T = fstride(NTR), TS_G = fstride(NV);
  // F^2 tiles (tendency): node (i, j, k) at i + Nq j + PS2 k.  At Nq = 5 a zeta-plane stride of 27 puts the 15 / 10
  // eta-lines of zeta-planes {0,1,2} / {3,4} into distinct banks (cm7_yline deals the lines to the lanes that way)
  static constexpr int PS2 = (Nq == 5) ? NF + 2 : NF;
  static constexpr int SLOT2 = (Nq - 1) * PS2 + NF;
  static constexpr int TEND_DOUBLES = (NV + 2 * NV + 1 + NV) * SLOT + NV * SLOT2 + 5 * TS_T + NTR * NF + TAIL;   // Q, F^1 F^3 (G lands there), c, residual, F^2, traces
  static constexpr int GRAD_DOUBLES = (NV + 3 * NS) * SLOT + 5 * TS_G + NV * NF + TAIL;            // Q (then s in place), ds/dxi_d, traces
  static_assert(2 * NV >= NG, "the packed SGS fluxes are staged in the F^1, F^3 tiles");
  static constexpr size_t TEND_SMEM = sizeof(double) * TEND_DOUBLES;
  static constexpr size_t GRAD_SMEM = sizeof(double) * GRAD_DOUBLES;
  static constexpr int fit(size_t smem) { return (int)(233472 / (smem + 1024)); }
  static constexpr int cap(int b, int hi) { return b < 1 ? 1 : (b > hi ? hi : b); }
#ifndef CM_T_REGTHREADS
#define CM_T_REGTHREADS 640
#endif
#ifndef CM_G_REGTHREADS
#define CM_G_REGTHREADS 896
#endif
  // 640: >= 100 registers per thread; the largest CTA that still fits twice (N = 6: 352 threads) is held to 93 registers
  static constexpr int MINB_T = cap(fit(TEND_SMEM), cap((THREADS > 320 && THREADS <= 352 ? 704 : CM_T_REGTHREADS) / THREADS, 16));
  static constexpr int MINB_G = cap(fit(GRAD_SMEM), cap(896 / THREADS, 16));   // >= 72 registers per thread
};

template <int Nq, int D> struct Cm7Str { static constexpr int value = (D == 0) ? 1 : (D == 1) ? Nq : Nq * Nq; };

// index into the packed SGS array (tau xx,yy,zz,xy,xz,yz | J+D x,y,z | d_q x,y,z) of the k-th value axis d needs
__host__ __device__ constexpr int cm7_gidx(int d, int k) {
  return (k == 3) ? 6 + d : (k == 4) ? 9 + d : (k == d) ? d : k + d + 2;   // (0,1)->3, (0,2)->4, (1,2)->5
}

// site (geopotential + reference column) from a z-table row held in shared memory
__device__ __forceinline__ void cm7_site(const double* zrow, CmSite& s) {
  s.Phi = zrow[0]; s.rho_r = zrow[1]; s.rhoe_r = zrow[2]; s.rhoq_r = zrow[3]; s.E_r = zrow[4]; s.q_r = zrow[5]; s.icvm_r = zrow[6]; s.taus = 0.0;
}

// primitives the gradient needs (u, v, w, h_tot, q): eq. (6)-(10), (13)-(14)
// RICH: also theta_v (eq. 40), stored behind the last regular gradient variable (index 5 moist, 4 dry)
template <bool MOIST, bool RICH = false>
__device__ __forceinline__ void cm7_eos_grad(const CmKP& p, const double* Y, double Phi, double* s) {
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
  if (RICH) s[MOIST ? 5 : 4] = cm_theta_v(th, pr, ir);
}

// ------------------------------------------------------------------------------------------------
// Position of the CTA's element in the tiled library order (cm_dg_lib.cu): the grid is (PY*L, Ez, (Ey/PY)*(Ex/L)) and
//   e = ((((ey / PY) * NXC + ex / L) * Ez + ez) * PY + ey % PY) * L + ex % L.
// ------------------------------------------------------------------------------------------------
struct Cm7Pos { int exl, eyl, ez, xc, yp, e, wallmask; };

__device__ __forceinline__ int cm7_divsmall(int a, int b, float invb) {   // a / b for 0 <= a < 2^22, exact
  int q = __float2int_rz(((float)a + 0.5f) * invb);
  const int r = a - q * b;
  if (r < 0) --q; else if (r >= b) ++q;
  return q;
}

__device__ __forceinline__ Cm7Pos cm7_position(const CmKP& p) {
  Cm7Pos q;
  const int bx = blockIdx.x, bz = blockIdx.z;
  q.eyl = cm7_divsmall(bx, p.gL, p.ginvL); q.exl = bx - q.eyl * p.gL;
  q.yp = cm7_divsmall(bz, p.gNXC, p.ginvNXC); q.xc = bz - q.yp * p.gNXC;
  q.ez = blockIdx.y;
  q.e = (bz * p.gEz + q.ez) * (p.gPY * p.gL) + bx;
  int m = 0;                                               // bit f set = face f of the element lies on a wall
  if (p.gbc[0]) { if (q.xc == 0 && q.exl == 0) m |= 1; if (q.xc == p.gNXC - 1 && q.exl == p.gL - 1) m |= 2; }
  if (p.gbc[1]) { if (q.yp == 0 && q.eyl == 0) m |= 4; if (q.yp == p.gNYP - 1 && q.eyl == p.gPY - 1) m |= 8; }
  if (p.gbc[2]) { if (q.ez == 0) m |= 16; if (q.ez == p.gEz - 1) m |= 32; }
  q.wallmask = m;
  return q;
}

// library index of the neighbour across face f = 2 d + s (periodic wrap; walls are flagged by wallmask)
__device__ __forceinline__ int cm7_neighbour(const CmKP& p, const Cm7Pos& q, int d, int s) {
  int lo = (d == 0) ? q.exl : (d == 1) ? q.eyl : q.ez;
  int hi = (d == 0) ? q.xc : (d == 1) ? q.yp : 0;
  const int nlo = (d == 0) ? p.gL : (d == 1) ? p.gPY : p.gEz;
  const int nhi = (d == 0) ? p.gNXC : (d == 1) ? p.gNYP : 1;
  lo += s ? 1 : -1;
  if (lo == nlo) { lo = 0; ++hi; } else if (lo < 0) { lo = nlo - 1; --hi; }
  if (hi == nhi) hi = 0; else if (hi < 0) hi = nhi - 1;
  const int exl = (d == 0) ? lo : q.exl, xc = (d == 0) ? hi : q.xc;
  const int eyl = (d == 1) ? lo : q.eyl, yp = (d == 1) ? hi : q.yp;
  const int ez = (d == 2) ? lo : q.ez;
  return (((yp * p.gNXC + xc) * p.gEz + ez) * p.gPY + eyl) * p.gL + exl;
}

// face node fn = f * NF + m  ->  face f = 2 d + s, own node nm, neighbour's coincident node np_
template <int Nq>
__device__ __forceinline__ void cm7_face_node(int fn, int& f, int& m, int& d, int& s, int& nm, int& np_, int& kline) {
  constexpr int NF = Nq * Nq, N = Nq - 1;
  f = fn / NF; m = fn - f * NF; d = f >> 1; s = f & 1;
  const int b = m / Nq, a = m - b * Nq;
  const int base = (d == 0) ? Nq * m : (d == 1) ? a + NF * b : m;
  const int span = N * ((d == 0) ? 1 : (d == 1) ? Nq : NF);
  nm = s ? base + span : base;
  np_ = s ? base : base + span;
  kline = b;                                               // zeta index of the node for d < 2
}

// CTA prologue shared by both kernels: z rows and neighbour traces to shared memory by cp.async.
//   T[f * TS + v * NF + m]: value v of the node of neighbour f that coincides with face node m of face f
template <int Nq, int NV, int NGD, int TS, int THREADS>
__device__ __forceinline__ void cm7_prefetch_traces(const CmKP& p, const Cm7Pos& q, int t, double* __restrict__ T,
                                                    double* __restrict__ zt) {
  constexpr int NF = Nq * Nq, NP = NF * Nq, ZR = Nq + 2;
  // group 0: z rows (phase 1 needs them)
  for (int c = t; c < ZR * 7; c += THREADS) {
    const int r = c / 7, col = c - 7 * r;
    int row = q.ez * Nq + r - 1;                                           // own rows; r = 0 / ZR-1: the facing rows below / above
    if (r == 0) row = (q.wallmask & 16) ? -1 : (q.ez > 0 ? row : p.gEz * Nq - 1);
    if (r == ZR - 1) row = (q.wallmask & 32) ? -1 : (q.ez < p.gEz - 1 ? row : 0);
    if (row >= 0) cm7_cp8(zt + r * CM_ZSM_W + col, p.ztab + (size_t)row * CM_ZTAB_W + col);
  }
  cm7_cp_commit();
  // group 1: neighbour traces (phase 2 needs them)
  for (int fn = THREADS - 1 - t; fn < 6 * NF; fn += THREADS) {   // the thread that will run the face task of node fn
    int f, m, d, s, nm, np_, kline;
    cm7_face_node<Nq>(fn, f, m, d, s, nm, np_, kline);
    if (!((q.wallmask >> f) & 1)) {
      const int nb = cm7_neighbour(p, q, d, s);
      const size_t idp = (size_t)nb * NP + np_;
      double* dst = T + f * TS + m;
      const double* src = p.Q + idp;
#pragma unroll
      for (int v = 0; v < NV; ++v) { cm7_cp8(dst + v * NF, src); src += p.stride; }
      if (NGD > 0) {
        const double* g = p.G + idp;
#pragma unroll
        for (int k = 0; k < NGD; ++k) cm7_cp8(dst + (NV + k) * NF, g + (size_t)cm7_gidx(d, k) * p.stride);
      }
    }
  }
  cm7_cp_commit();
}

// ------------------------------------------------------------------------------------------------
// tendency, phase 2a: face task.  Replaces the trace of face node fn by
//   rf[v] = -(1/2) sJ n.F^+[v] - (1/2) sJ lambda (Y^-[v] - Y^+[v])          interior / periodic (eq. 27 with R1, R2, R6)
//   rf    = [0; -(p' + rho u_n (u_n + lambda)) sJ n; 0; 0] (+ sJ SHF on the bottom wall)   free-slip wall (A6-A7, R10)
// so that  sJ (n.F^- - F*) = ch * sJ n.F^- + rf  with ch = 1/2 (interior) or 1 (wall); the line task adds the ch term.
// ------------------------------------------------------------------------------------------------
template <int Nq, bool MOIST, bool SGS>
__device__ __forceinline__ void cm7_tend_face(const CmKP& p, const double* __restrict__ Qs, const double* __restrict__ cs,
                                              double* __restrict__ T, const double* __restrict__ zt, int wallmask, int fn) {
  using C = CmCfg7<Nq, MOIST>;
  constexpr int NF = C::NF, NV = C::NV, NGD = C::NGD, SLOT = C::SLOT, TS = C::TS_T;
  int f, m, d, s, nm, np_, kline;
  cm7_face_node<Nq>(fn, f, m, d, s, nm, np_, kline);
  const bool wall = (wallmask >> f) & 1;
  double* tr = T + f * TS + m;
  const double sgn = s ? 1.0 : -1.0;
  const double sJ = (d == 0) ? p.cA[0] : (d == 1) ? p.cA[1] : p.cA[2];
  const double A = sgn * sJ;
  double Ym[6];
#pragma unroll
  for (int v = 0; v < NV; ++v) Ym[v] = Qs[v * SLOT + nm];
  const double cm_ = cs[nm];
  const double mn = (d == 0) ? Ym[1] : (d == 1) ? Ym[2] : Ym[3];
  const double unm = sgn * (mn * cm_rcp(Ym[0]));                            // u^- . n
  double rf[6];
  CmSite st; CmPrim P;
  if (!wall) {
    double Yp[6], gp[5];
#pragma unroll
    for (int v = 0; v < NV; ++v) Yp[v] = tr[v * NF];
    if (SGS)
#pragma unroll
      for (int k = 0; k < NGD; ++k) gp[k] = tr[(NV + k) * NF];
    cm7_site(zt + ((d < 2) ? 1 + kline : (s ? Nq + 1 : 0)) * CM_ZSM_W, st);
    cm_eos<MOIST>(p, Yp, st, P);
    const double ud = (d == 0) ? P.u : (d == 1) ? P.v : P.w;
    double wA = ud, t0 = 0.0, t1 = 0.0, t2 = 0.0, eA = 0.0, dqA = 0.0;
    if (SGS) {
      t0 = gp[0]; t1 = gp[1]; t2 = gp[2];
      eA = t0 * P.u + t1 * P.v + t2 * P.w + gp[3];
      if (MOIST) { dqA = gp[4]; wA += dqA; }
    }
    double Fp[6];
    Fp[0] = Yp[0] * wA;
    Fp[1] = Yp[1] * wA + ((d == 0) ? P.pp : 0.0) + Yp[0] * t0;
    Fp[2] = Yp[2] * wA + ((d == 1) ? P.pp : 0.0) + Yp[0] * t1;
    Fp[3] = Yp[3] * wA + ((d == 2) ? P.pp : 0.0) + Yp[0] * t2;
    Fp[4] = (Yp[4] + P.p) * ud + Yp[0] * eA;
    if (MOIST) Fp[5] = Yp[5] * ud + Yp[0] * dqA;
    const double cp = cm_sqrt(P.c2);
    const double lam = fmax(fabs(unm) + cm_, fabs(ud) + cp);               // lambda (R2)
    const double hA = -0.5 * A, hl = -0.5 * (lam * sJ);
#pragma unroll
    for (int v = 0; v < NV; ++v) rf[v] = hA * Fp[v] + hl * (Ym[v] - Yp[v]);
  } else {
    cm7_site(zt + ((d < 2) ? 1 + kline : (s ? Nq : 1)) * CM_ZSM_W, st);
    cm_eos<MOIST>(p, Ym, st, P);
    const double lam = fabs(unm) + cm_;
    const double mom = -(P.pp + Ym[0] * unm * (unm + lam)) * A;
#pragma unroll
    for (int v = 0; v < NV; ++v) rf[v] = 0.0;
    rf[1] = (d == 0) ? mom : 0.0; rf[2] = (d == 1) ? mom : 0.0; rf[3] = (d == 2) ? mom : 0.0;
    if (f == 4) {                                                          // prescribed surface fluxes, drag law (App. A1)
      const double Aw[3] = {0.0, 0.0, -sJ};
      cm_surface_flux<MOIST>(p, Aw, sJ, Ym[0], Qs + nm + NF, SLOT, rf);
    }
  }
#pragma unroll
  for (int v = 0; v < NV; ++v) tr[v * NF] = rf[v];
}

// eta-line l -> first node in an F^2 tile; false = idle lane.  Nq = 5: lanes 0..14 hold zeta-planes 0..2, lanes 16..25
// planes 3..4 (see CmCfg7::PS2)
template <int Nq>
__device__ __forceinline__ bool cm7_yline(int l, int& base) {
  constexpr int NF = Nq * Nq, PS2 = (Nq == 5) ? NF + 2 : NF;
  if (Nq == 5) {
    if (l == 15 || l >= 26) return false;
    const int ll = (l < 15) ? l : l - 1;              // 0..24
    const int b = ll / 5, a = ll - 5 * b;
    base = a + PS2 * b;
    return true;
  }
  if (l >= NF) return false;
  const int b = l / Nq, a = l - b * Nq;
  base = a + PS2 * b;
  return true;
}

// tendency, phase 2b: line task.  q0 = first node of the line in the first of the NV tiles holding F^D (tile stride
// TSL, node stride STR); on return the line holds D_D F^D minus the lifted own-side half of the face term at its two
// ends (eq. 32)
template <int Nq, int NV, int TSL, int STR, int D>
__device__ __forceinline__ void cm7_tend_line(const CmKP& p, double* __restrict__ q0, int wallmask) {
  constexpr int N = Nq - 1;
  const double c0 = p.inv_w0 * (((wallmask >> (2 * D)) & 1) ? 1.0 : 0.5);      // -sgn = +1 at the low end
  const double cN = -p.inv_w0 * (((wallmask >> (2 * D + 1)) & 1) ? 1.0 : 0.5);
  constexpr int LU = CM_LINE_UNROLL;
#pragma unroll LU
  for (int v = 0; v < NV; ++v) {
    double* q = q0 + v * TSL;
    double x[Nq], y[Nq];
#pragma unroll
    for (int m = 0; m < Nq; ++m) x[m] = q[m * STR];
#pragma unroll
    for (int i = 0; i < Nq; ++i) {
      double s = 0.0;
#pragma unroll
      for (int m = 0; m < Nq; ++m) s += p.D[i][m] * x[m];
      y[i] = s;
    }
    y[0] += c0 * x[0];
    y[N] += cN * x[N];
#pragma unroll
    for (int i = 0; i < Nq; ++i) q[i * STR] = y[i];
  }
}

// MODE: 0 dQ := rhs | 1 LSRK stage reading the residual | 2 LSRK stage with A_s = 0 (residual not read)
template <int Nq, bool MOIST, bool SGS, int MODE>
__global__ void __launch_bounds__(CmCfg7<Nq, MOIST>::THREADS, CmCfg7<Nq, MOIST>::MINB_T) cm7_tendency_kernel(const __grid_constant__ CmKP p) {
  using C = CmCfg7<Nq, MOIST>;
  constexpr int NF = C::NF, NP = C::NP, N = Nq - 1, NV = C::NV, NG = C::NG, SLOT = C::SLOT, NFP = C::NFP, THREADS = C::THREADS;
  constexpr int TS = C::TS_T;
  extern __shared__ __align__(128) double smem7[];
  double* Qt = smem7;                                  // [NV][SLOT]     state
  double* Ft = Qt + NV * SLOT;                         // [2][NV][SLOT]  F^1, F^3 (the packed SGS fluxes G land here)
  double* ct = Ft + 2 * NV * SLOT;                     // [SLOT]         sound speed
  double* Rt = ct + SLOT;                              // [NV][SLOT]     LSRK residual
  double* F2 = Rt + NV * SLOT;                         // [NV][SLOT2]    F^2 (zeta-plane stride PS2)
  double* T = F2 + NV * C::SLOT2;                          // [6][TS]        neighbour traces [v][m] per face, then rf
  double* zt = T + 5 * TS + C::NTR * NF;      // [ZR][CM_ZSM_W]
  uint64_t* mbar = reinterpret_cast<uint64_t*>(zt + (C::ZR - 1) * CM_ZSM_W + 7);

  const int t = threadIdx.x;
  const Cm7Pos pos = cm7_position(p);
  const int e = pos.e;
  const int sh = C::ODD ? (e & 1) : 0;

  if (t == THREADS - 32) { cm7_mbar_init(mbar, 1); cm7_fence_mbar_init(); }
  __syncthreads();                                     // mbarrier initialised: from here on nobody waits for an instruction
                                                       // stream of another warp, only for data
  if (t == THREADS - 32) {                             // lane 0 of the last warp issues the bulk copies
    const long long src = (long long)e * NP - sh;
    const uint32_t mb = cm7_saddr(mbar);
    cm7_mbar_expect_tx(mbar, (uint32_t)((NV + (SGS ? NG : 0) + (MODE == 1 ? NV : 0)) * SLOT * sizeof(double)));
    {
      const double* g = p.Q + src; uint32_t d = cm7_saddr(Qt);
#pragma unroll
      for (int v = 0; v < NV; ++v) { cm7_bulk_g2s_raw(d, g, SLOT * 8, mb); g += p.stride; d += SLOT * 8; }
    }
    if (SGS) {
      const double* g = p.G + src; uint32_t d = cm7_saddr(Ft);
#pragma unroll
      for (int k = 0; k < NG; ++k) { cm7_bulk_g2s_raw(d, g, SLOT * 8, mb); g += p.stride; d += SLOT * 8; }
    }
    if (MODE == 1) {
      const double* g = p.dQ + src; uint32_t d = cm7_saddr(Rt);
#pragma unroll
      for (int v = 0; v < NV; ++v) { cm7_bulk_g2s_raw(d, g, SLOT * 8, mb); g += p.stride; d += SLOT * 8; }
    }
  } else if (t > THREADS - 32 && p.ahead > 0 && e + p.ahead < p.Ne) {
    // the other lanes of that warp pull the tiles of the element `ahead` places further on in the launch order into L2:
    // its own bulk copies and the trace gathers of its neighbours then hit L2 instead of waiting on DRAM
    constexpr int NTILE = NV + (SGS ? NG : 0) + (MODE == 1 ? NV : 0);
    const int ea = e + p.ahead;
    const long long src = (long long)ea * NP - (C::ODD ? (ea & 1) : 0);
    for (int j = t - (THREADS - 32) - 1; j < NTILE; j += 31) {
      const bool isq = j < NV, isg = SGS && !isq && j < NV + NG;
      const int idx = isq ? j : isg ? j - NV : j - NV - (SGS ? NG : 0);
      const double* g = isq ? p.Q : isg ? p.G : p.dQ;
      cm7_prefetch_l2(g + (size_t)idx * p.stride + src, SLOT * 8);
    }
  }
  cm7_prefetch_traces<Nq, NV, SGS ? C::NGD : 0, TS, THREADS>(p, pos, t, T, zt);

  double* Qs = Qt + sh; double* Fs = Ft + sh; double* cs = ct + sh; const double* Rs = Rt + sh;
  const int n = t;
  const bool node = t < NP;
  const int k_ = n / NF, j_ = (n - k_ * NF) / Nq, i_ = n - k_ * NF - j_ * Nq;
  const int n2 = n + (C::PS2 - NF) * k_;               // index in the F^2 tiles
  CmSite st;                                           // own row of the z table through the read-only path (L1-resident): the
  if (node) {                                          // shared-memory copy of the z rows is only needed by the face tasks
    const double2* zr = reinterpret_cast<const double2*>(p.ztab + (size_t)(pos.ez * Nq + k_) * CM_ZTAB_W);
    const double2 a = __ldg(zr), b = __ldg(zr + 1), c = __ldg(zr + 2), d = __ldg(zr + 3);
    st.Phi = a.x; st.rho_r = a.y; st.rhoe_r = b.x; st.rhoq_r = b.y; st.E_r = c.x; st.q_r = c.y; st.icvm_r = d.x; st.taus = d.y;
  }
  cm7_mbar_wait(mbar, 0);

  // ---- phase 1: primitives and contravariant fluxes of the own node (F^1, F^2 overwrite G in place)
  double buoy = 0.0;
  double Y[6];                                         // the node's state stays in registers until the update in phase 3
  if (node) {
    double g[12]; CmPrim P;
#pragma unroll
    for (int v = 0; v < NV; ++v) Y[v] = Qs[v * SLOT + n];
    if (SGS)
#pragma unroll
      for (int k = 0; k < NG; ++k) g[k] = Fs[k * SLOT + n];
    cm_eos<MOIST>(p, Y, st, P);
    buoy = P.drho * p.th.grav;
    cs[n] = cm_sqrt(P.c2);
    double Fa[6], Fb[6], Fc[6];
    cm_flux_axis<MOIST, 0>(Y, P, SGS, g, p.cA[0], Fa);
    cm_flux_axis<MOIST, 1>(Y, P, SGS, g, p.cA[1], Fb);
    cm_flux_axis<MOIST, 2>(Y, P, SGS, g, p.cA[2], Fc);
#pragma unroll
    for (int v = 0; v < NV; ++v) { Fs[v * SLOT + n] = Fa[v]; Fs[(NV + v) * SLOT + n] = Fc[v]; F2[v * C::SLOT2 + n2] = Fb[v]; }
  }
  cm7_cp_wait_but_one();                               // this thread's z-row copies have landed
  __syncthreads();                                     // fluxes, sound speed and z rows visible

  // ---- phase 2: line tasks (one warp per direction), then face tasks (from the last thread downwards: the warp
  // without line tasks takes the second round).  Independent of each other; a face task needs only the traces its own
  // thread has copied, so the wait for them sits behind the line task and no CTA barrier is needed for the traces
  for (int lt = t; lt < 3 * NFP; lt += THREADS) {
    const int d = lt / NFP, l = lt % NFP;
    if (d == 0) { if (l < NF) cm7_tend_line<Nq, NV, SLOT, 1, 0>(p, Fs + Nq * l, pos.wallmask); }
    else if (d == 1) { int base; if (cm7_yline<Nq>(l, base)) cm7_tend_line<Nq, NV, C::SLOT2, Nq, 1>(p, F2 + base, pos.wallmask); }
    else { if (l < NF) cm7_tend_line<Nq, NV, SLOT, NF, 2>(p, Fs + NV * SLOT + l, pos.wallmask); }
  }
  cm7_cp_wait_all();                                   // this thread's trace copies have landed
  for (int fn = THREADS - 1 - t; fn < 6 * NF; fn += THREADS) cm7_tend_face<Nq, MOIST, SGS>(p, Qs, cs, T, zt, pos.wallmask, fn);
  __syncthreads();

  // ---- phase 3: assemble the tendency of the own node and update
  if (node) {
    double acc[6], lift[6], Yo[6], Ro[6];
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      acc[v] = Fs[v * SLOT + n] + F2[v * C::SLOT2 + n2] + Fs[(NV + v) * SLOT + n];
      lift[v] = 0.0;
      if (MODE != 0) Yo[v] = Y[v];
      if (MODE == 1) Ro[v] = Rs[v * SLOT + n];
    }
    // rf of the faces the node lies on
    const int c3[3] = {i_, j_, k_};
    const int m3[3] = {j_ + Nq * k_, i_ + Nq * k_, i_ + Nq * j_};
#pragma unroll
    for (int d = 0; d < 3; ++d)
      if (c3[d] == 0 || c3[d] == N) {
        const double* tr = T + (2 * d + (c3[d] == N ? 1 : 0)) * TS + m3[d];
#pragma unroll
        for (int v = 0; v < NV; ++v) lift[v] += tr[v * NF];
      }
    const size_t idx = (size_t)e * NP + n;
    double* o1 = p.dQ + idx;
    double* o2 = p.Qnew + idx;
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      double rhs = -p.invJ * (acc[v] - p.inv_w0 * lift[v]);
      if (v == 3) rhs -= buoy;                                   // -(rho - rho_r) grad Phi   (eq. 4)
      if (v >= 1 && v <= 3) rhs -= st.taus * (Y[v] - Y[0] * p.urelax[v - 1]);   // Rayleigh sponge (A4); tau_s = 0 outside the layer
      if (MODE == 0) {
        __stcs(o1, rhs);
      } else {
        // a5: dU <- A_s dU + dt RHS ; U <- U + B_s dU
        const double dnew = (MODE == 1) ? p.rka * Ro[v] + p.dt * rhs : p.dt * rhs;
        __stcs(o1, dnew);
        __stcs(o2, Yo[v] + p.rkb * dnew);
        o2 += p.stride;
      }
      o1 += p.stride;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// a2: auxiliary gradient + Smagorinsky-Lilly (flat bricks), same decomposition
// ------------------------------------------------------------------------------------------------
// face task: trace -> s* - s^- (eq. 30-31: central flux; walls A6, A8)
template <int Nq, bool MOIST>
__device__ __forceinline__ void cm7_grad_face(const CmKP& p, const double* __restrict__ ss, double* __restrict__ T,
                                              const double* __restrict__ zt, int wallmask, int fn) {
  using C = CmCfg7<Nq, MOIST>;
  constexpr int NF = C::NF, NV = C::NV, NS = C::NS, SLOT = C::SLOT, TS = C::TS_G;
  int f, m, d, s, nm, np_, kline;
  cm7_face_node<Nq>(fn, f, m, d, s, nm, np_, kline);
  double* tr = T + f * TS + m;
  double dl[5];
  if (!((wallmask >> f) & 1)) {
    double Yp[6], sp[5];
#pragma unroll
    for (int v = 0; v < NV; ++v) Yp[v] = tr[v * NF];
    cm7_eos_grad<MOIST>(p, Yp, zt[((d < 2) ? 1 + kline : (s ? Nq + 1 : 0)) * CM_ZSM_W], sp);
#pragma unroll
    for (int v = 0; v < NS; ++v) dl[v] = 0.5 * (sp[v] - ss[v * SLOT + nm]);
  } else {
    // wall: u_bc = u^- - (n.u^-) n  (A6); scalars unchanged (A8)
#pragma unroll
    for (int v = 0; v < NS; ++v) dl[v] = (v == d) ? -ss[v * SLOT + nm] : 0.0;
  }
#pragma unroll
  for (int v = 0; v < NS; ++v) tr[v * NF] = dl[v];
}

template <int Nq, bool MOIST, int D>
__device__ __forceinline__ void cm7_grad_line(const CmKP& p, const double* __restrict__ ss, double* __restrict__ dd, int l) {
  using C = CmCfg7<Nq, MOIST>;
  constexpr int NF = C::NF, NS = C::NS, SLOT = C::SLOT, STR = Cm7Str<Nq, D>::value, OSTR = (D == 2) ? NF : 1;
  const int b = l / Nq, a = l - b * Nq;
  const int base = (D == 0) ? Nq * l : (D == 1) ? a + NF * b : l;
  const int obase = (D == 2) ? l : Nq * l;              // eta-derivatives are stored with i and j swapped (contiguous)
#pragma unroll
  for (int v = 0; v < NS; ++v) {
    const double* in = ss + v * SLOT + base;
    double* out = dd + v * SLOT + obase;
    double x[Nq];
#pragma unroll
    for (int m = 0; m < Nq; ++m) x[m] = in[m * STR];
#pragma unroll
    for (int i = 0; i < Nq; ++i) {
      double s = 0.0;
#pragma unroll
      for (int m = 0; m < Nq; ++m) s += p.D[i][m] * x[m];
      out[i * OSTR] = s;
    }
  }
}

// RAW: false packed SGS fluxes (hot path) | true the 15 raw gradients (cm_dg_gradient)
// GEM: the packed SGS fluxes are stored element-major, G[e][NG][SLOT] (one bulk copy per element for the row-sweep
// tendency kernel), instead of field-major G[k][stride]
template <int Nq, bool MOIST, bool RAW, bool GEM = false>
__global__ void __launch_bounds__(CmCfg7<Nq, MOIST>::THREADS, CmCfg7<Nq, MOIST>::MINB_G) cm7_gradient_kernel(const __grid_constant__ CmKP p) {
  using C = CmCfg7<Nq, MOIST>;
  constexpr int NF = C::NF, NP = C::NP, N = Nq - 1, NV = C::NV, NS = C::NS, SLOT = C::SLOT, NFP = C::NFP, THREADS = C::THREADS;
  constexpr int TS = C::TS_G;
  extern __shared__ __align__(128) double smem7[];
  double* Qt = smem7;                                  // [NV][SLOT]      state, then the gradient variables in place
  double* dt_ = Qt + NV * SLOT;                        // [3][NS][SLOT]   reference-space derivatives
  double* T = dt_ + 3 * NS * SLOT;                     // [6][TS]         neighbour traces [v][m] per face, then s* - s^-
  double* zt = T + 5 * TS + NV * NF;              // [ZR][CM_ZSM_W]
  uint64_t* mbar = reinterpret_cast<uint64_t*>(zt + (C::ZR - 1) * CM_ZSM_W + 7);

  const int t = threadIdx.x;
  const Cm7Pos pos = cm7_position(p);
  const int e = pos.e;
  const int sh = C::ODD ? (e & 1) : 0;
  if (t == THREADS - 32) {
    cm7_mbar_init(mbar, 1);
    cm7_fence_mbar_init();
    const long long src = (long long)e * NP - sh;
    cm7_mbar_expect_tx(mbar, (uint32_t)(NV * SLOT * sizeof(double)));
#pragma unroll
    for (int v = 0; v < NV; ++v) cm7_bulk_g2s(Qt + v * SLOT, p.Q + v * p.stride + src, SLOT * 8, mbar);
  } else if (t > THREADS - 32 && t <= THREADS - 32 + NV && p.ahead > 0 && e + p.ahead < p.Ne) {
    const int ea = e + p.ahead, v = t - (THREADS - 32) - 1;   // L2 prefetch one wave ahead (see the tendency kernel)
    cm7_prefetch_l2(p.Q + (size_t)v * p.stride + ((long long)ea * NP - (C::ODD ? (ea & 1) : 0)), SLOT * 8);
  }
  cm7_prefetch_traces<Nq, NV, 0, TS, THREADS>(p, pos, t, T, zt);
  double* ss = Qt + sh; double* dd = dt_ + sh;
  const int n = t;
  const bool node = t < NP;
  const int k_ = n / NF, j_ = (n - k_ * NF) / Nq, i_ = n - k_ * NF - j_ * Nq;
  const int nT = j_ + Nq * i_ + NF * k_;               // index in the eta-derivative tiles (i, j swapped)
  cm7_cp_wait_but_one();
  __syncthreads();
  cm7_mbar_wait(mbar, 0);

  // ---- phase 1: gradient variables of the own node, in place of the state
  if (node) {
    double Y[6], s[5];
#pragma unroll
    for (int v = 0; v < NV; ++v) Y[v] = ss[v * SLOT + n];
    cm7_eos_grad<MOIST>(p, Y, zt[(1 + k_) * CM_ZSM_W], s);
#pragma unroll
    for (int v = 0; v < NS; ++v) ss[v * SLOT + n] = s[v];
  }
  cm7_cp_wait_all();
  __syncthreads();

  // ---- phase 2: face tasks and line tasks, independent
  for (int fn = THREADS - 1 - t; fn < 6 * NF; fn += THREADS) cm7_grad_face<Nq, MOIST>(p, ss, T, zt, pos.wallmask, fn);
  for (int lt = t; lt < 3 * NFP; lt += THREADS) {
    const int d = lt / NFP, l = lt % NFP;
    if (l < NF) {
      if (d == 0) cm7_grad_line<Nq, MOIST, 0>(p, ss, dd, l);
      else if (d == 1) cm7_grad_line<Nq, MOIST, 1>(p, ss, dd + NS * SLOT, l);
      else cm7_grad_line<Nq, MOIST, 2>(p, ss, dd + 2 * NS * SLOT, l);
    }
  }
  __syncthreads();

  // ---- phase 3: lifted jumps, physical gradient, closure, store
  if (node) {
    const size_t idx = (size_t)e * NP + n;
    double Gr[5][3];
    const int c3[3] = {i_, j_, k_};
    const int m3[3] = {j_ + Nq * k_, i_ + Nq * k_, i_ + Nq * j_};
#pragma unroll
    for (int c = 0; c < 3; ++c) {
#pragma unroll
      for (int v = 0; v < NS; ++v) Gr[v][c] = dd[(c * NS + v) * SLOT + (c == 1 ? nT : n)];
      if (c3[c] == 0 || c3[c] == N) {
        const bool hi = (c3[c] == N);
        const double* tr = T + (2 * c + (hi ? 1 : 0)) * TS + m3[c];
        const double w = hi ? p.inv_w0 : -p.inv_w0;
#pragma unroll
        for (int v = 0; v < NS; ++v) Gr[v][c] += w * tr[v * NF];
      }
#pragma unroll
      for (int v = 0; v < NS; ++v) Gr[v][c] *= (p.cA[c] * p.invJ);
    }
    if (!MOIST) { Gr[4][0] = Gr[4][1] = Gr[4][2] = 0.0; }
    double* o = (GEM && !RAW) ? p.Gout + (size_t)e * (C::NG * SLOT) + n : p.Gout + idx;
    const long long st = (GEM && !RAW) ? (long long)SLOT : p.stride;
    if (RAW) {
#pragma unroll
      for (int v = 0; v < 5; ++v)
#pragma unroll
        for (int c = 0; c < 3; ++c) __stcs(o + (size_t)(3 * v + c) * st, Gr[v][c]);
    } else {
      // eq. (33)-(39): closure (cm_closure; the Richardson factor needs theta_v and is served by the other gradient
      // kernels: cm_dg_setup routes richardson = 1 at these orders to the thread-per-node kernels)
      double g[12];
      cm_closure<MOIST>(p, Gr, p.cs2delta2, p.d2[0], p.d2[1], p.d2[2], 1.0, 0.0, g);
#pragma unroll
      for (int k = 0; k < C::NG; ++k) o[k * st] = g[k];
    }
  }
}

// ------------------------------------------------------------------------------------------------
// a2, second form (used when every line task has its own thread, 3 * NFP <= THREADS): the line task owns the face
// terms of its two end nodes.  Its 2 x NV neighbour-trace values are loaded into REGISTERS at CTA start (the addresses
// follow from blockIdx, so the loads are in flight together with the bulk TMA of the element's own tiles) and are
// consumed only in phase 2: no trace buffer, no cp.async, no second pass over the face nodes, and the lifted jumps
// are folded into the line's end values -- half the shared-memory traffic of cm7_gradient_kernel (profiles/r1e_v9.md:
// that kernel kept the shared-memory data pipe 78 % busy).
// ------------------------------------------------------------------------------------------------
template <int Nq, bool MOIST> struct CmCfg9 {
  using C7 = CmCfg7<Nq, MOIST>;
  static constexpr int GRAD_DOUBLES = (C7::NV + 3 * C7::NS + 1) * C7::SLOT + 2;   // Q (then s in place), ds/dxi_d, d theta_v/d zeta (eq. 40), mbarrier
  static constexpr size_t GRAD_SMEM = sizeof(double) * GRAD_DOUBLES;
  static constexpr bool OK = 3 * C7::NFP <= C7::THREADS;
  static constexpr int MINB_G = C7::cap(C7::fit(GRAD_SMEM), C7::cap(CM_G_REGTHREADS / C7::THREADS, 16));   // 896: >= 72 registers per thread
};

// line l of direction D -> first node and zeta index.  For Nq = 5 the eta-lines are dealt to the lanes so that each
// half-warp holds whole zeta-planes {0, 1, 4} and {2, 3}: the 25-double plane stride then costs one 2-way bank
// conflict instead of two (lanes 15 and 26..31 idle).
template <int Nq, int D>
__device__ __forceinline__ bool cm9_line(int l, int& base, int& kline) {
  constexpr int NF = Nq * Nq;
  if (D == 1 && Nq == 5) {
    int a, b;
    if (l < 10) { b = l / 5; a = l - 5 * b; }
    else if (l < 15) { b = 4; a = l - 10; }
    else if (l >= 16 && l < 26) { b = 2 + (l - 16) / 5; a = (l - 16) % 5; }
    else return false;
    base = a + NF * b; kline = b;
    return true;
  }
  if (l >= NF) return false;
  const int b = l / Nq, a = l - b * Nq;
  base = (D == 0) ? Nq * l : (D == 1) ? a + NF * b : l;
  kline = b;
  return true;
}

template <int Nq, bool MOIST, int D, bool RICH>
__device__ __forceinline__ void cm9_grad_line(const CmKP& p, const double* __restrict__ ss, double* __restrict__ dd,
                                              const double (&Yp)[2][6], const double (&Php)[2], int wallmask, int base) {
  using C = CmCfg7<Nq, MOIST>;
  // theta_v (eq. 40) needs its vertical derivative only: on flat bricks that is the zeta line
  constexpr int N = Nq - 1, NS = C::NS + ((RICH && D == 2) ? 1 : 0), SLOT = C::SLOT, STR = Cm7Str<Nq, D>::value;
  double dl[2][6];                                      // s* - s^- at the two ends (eq. 30-31: central flux)
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    const int nm = s ? base + N * STR : base;
    if (!((wallmask >> (2 * D + s)) & 1)) {
      double sp[6];
      cm7_eos_grad<MOIST, (RICH && D == 2)>(p, Yp[s], Php[s], sp);
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

// RICH: theta_v is a further gradient variable (its zeta derivative feeds the stability factor f_b of eq. 40)
template <int Nq, bool MOIST, bool RAW, bool GEM = false, bool RICH = false>
__global__ void __launch_bounds__(CmCfg7<Nq, MOIST>::THREADS, CmCfg9<Nq, MOIST>::MINB_G) cm9_gradient_kernel(const __grid_constant__ CmKP p) {
  using C = CmCfg7<Nq, MOIST>;
  constexpr int NF = C::NF, NP = C::NP, N = Nq - 1, NV = C::NV, NS = C::NS, SLOT = C::SLOT, NFP = C::NFP, THREADS = C::THREADS;
  extern __shared__ __align__(128) double smem7[];
  double* Qt = smem7;                                  // [NV][SLOT]      state, then the gradient variables in place
  double* dt_ = Qt + NV * SLOT;                        // [3][NS][SLOT] (+1) reference-space derivatives + lifted jumps
  uint64_t* mbar = reinterpret_cast<uint64_t*>(dt_ + (3 * NS + 1) * SLOT);

  const int t = threadIdx.x;
  const Cm7Pos pos = cm7_position(p);
  const int e = pos.e;
  const int sh = C::ODD ? (e & 1) : 0;
  if (t == THREADS - 32) {
    cm7_mbar_init(mbar, 1);
    cm7_fence_mbar_init();
    const long long src = (long long)e * NP - sh;
    cm7_mbar_expect_tx(mbar, (uint32_t)(NV * SLOT * sizeof(double)));
#pragma unroll
    for (int v = 0; v < NV; ++v) cm7_bulk_g2s(Qt + v * SLOT, p.Q + v * p.stride + src, SLOT * 8, mbar);
  } else if (t > THREADS - 32 && t <= THREADS - 32 + NV && p.ahead > 0 && e + p.ahead < p.Ne) {
    // L2 prefetch of the state tiles of the element `ahead` places further on in the launch order (see the tendency kernel)
    const int ea = e + p.ahead, v = t - (THREADS - 32) - 1;
    cm7_prefetch_l2(p.Q + (size_t)v * p.stride + ((long long)ea * NP - (C::ODD ? (ea & 1) : 0)), SLOT * 8);
  }

  // ---- the thread's line task and the neighbour traces of its two end nodes, into registers
  const int d = t / NFP, l = t - d * NFP;
  int base = 0, kline = 0;
  bool line = false;
  if (d == 0) line = cm9_line<Nq, 0>(l, base, kline);
  else if (d == 1) line = cm9_line<Nq, 1>(l, base, kline);
  else if (d == 2) line = cm9_line<Nq, 2>(l, base, kline);
  double Yp[2][6], Php[2];
#pragma unroll
  for (int s = 0; s < 2; ++s) {
#pragma unroll
    for (int v = 0; v < 6; ++v) Yp[s][v] = 1.0;
    Php[s] = 0.0;
  }
  if (line) {
    const int span = N * ((d == 0) ? 1 : (d == 1) ? Nq : NF);
#pragma unroll
    for (int s = 0; s < 2; ++s)
      if (!((pos.wallmask >> (2 * d + s)) & 1)) {
        const double* src = p.Q + (size_t)cm7_neighbour(p, pos, d, s) * NP + (s ? base : base + span);
#pragma unroll
        for (int v = 0; v < NV; ++v) { Yp[s][v] = __ldg(src); src += p.stride; }
        int row = pos.ez * Nq + kline;                                   // d < 2: the neighbour node is at the same height
        if (d == 2) row = s ? ((pos.ez + 1 == p.gEz) ? 0 : (pos.ez + 1) * Nq) : ((pos.ez == 0 ? p.gEz : pos.ez) * Nq - 1);
        Php[s] = __ldg(p.ztab + (size_t)row * CM_ZTAB_W);
      }
  }

  double* ss = Qt + sh; double* dd = dt_ + sh;
  const int n = t;
  const bool node = t < NP;
  double Phi = 0.0;
  if (node) Phi = __ldg(p.ztab + (size_t)(pos.ez * Nq + n / NF) * CM_ZTAB_W);
  __syncthreads();                                     // mbarrier init visible
  cm7_mbar_wait(mbar, 0);

  // ---- phase 1: gradient variables of the own node, in place of the state
  if (node) {
    double Y[6], s[6];
#pragma unroll
    for (int v = 0; v < NV; ++v) Y[v] = ss[v * SLOT + n];
    cm7_eos_grad<MOIST, RICH>(p, Y, Phi, s);
#pragma unroll
    for (int v = 0; v < NS + (RICH ? 1 : 0); ++v) ss[v * SLOT + n] = s[v];
  }
  __syncthreads();

  // ---- phase 2: one thread per line: contraction + lifted jumps at its two ends
  if (line) {
    if (d == 0) cm9_grad_line<Nq, MOIST, 0, RICH>(p, ss, dd, Yp, Php, pos.wallmask, base);
    else if (d == 1) cm9_grad_line<Nq, MOIST, 1, RICH>(p, ss, dd + NS * SLOT, Yp, Php, pos.wallmask, base);
    else cm9_grad_line<Nq, MOIST, 2, RICH>(p, ss, dd + 2 * NS * SLOT, Yp, Php, pos.wallmask, base);
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
    double* o = (GEM && !RAW) ? p.Gout + (size_t)e * (C::NG * SLOT) + n : p.Gout + idx;
    const long long st = (GEM && !RAW) ? (long long)SLOT : p.stride;
    if (RAW) {
#pragma unroll
      for (int v = 0; v < 5; ++v)
#pragma unroll
        for (int c = 0; c < 3; ++c) __stcs(o + (size_t)(3 * v + c) * st, Gr[v][c]);
    } else {
      // eq. (33)-(40): closure (cm_closure); store tau, J + D, d_q
      double thv = 1.0, dthv = 0.0;
      if (RICH) { thv = ss[NS * SLOT + n]; dthv = (p.cA[2] * p.invJ) * dd[(3 * NS) * SLOT + n]; }
      double g[12];
      cm_closure<MOIST>(p, Gr, p.cs2delta2, p.d2[0], p.d2[1], p.d2[2], thv, dthv, g);
#pragma unroll
      for (int k = 0; k < C::NG; ++k) o[k * st] = g[k];
    }
  }
}
