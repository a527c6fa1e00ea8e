// cm_dg_kernels10.cuh -- ROW-SWEEP kernels for flat bricks (GEOM == 0): one CTA walks along a row of S x-adjacent
// elements, one element per iteration, and keeps a software pipeline of bulk-TMA loads one element ahead.
//
// Why (profiles/r1f_prefetch.md, profiles/r2_*.md): the CTA-per-element kernels of cm_dg_kernels7.cuh are bound by
// the load/store path of the SM, and the dearest part of it is the exchange of neighbour traces across the xi faces --
// 8-byte gathers with a 40-byte stride, one 32-byte sector and one L1 tag lookup per value.  In a row sweep the xi
// neighbours of an element are the CTA's own previous and next element:
//   * the tile of element it+1 is fetched (1-D bulk TMA, mbarrier complete_tx) while element it is computed -- it is
//     needed at the top of the next iteration anyway, so the xi+ face of element it reads its i = 0 plane straight from
//     that landed tile: no gather, no extra traffic;
//   * the xi- face reads the i = N plane of element it-1, which phase 1 of that element saved (state + the SGS values
//     the x-normal flux needs) in a small carry buffer;
//   * only the two ends of the row gather xi traces from global memory (1/S of the faces), eta and zeta traces are
//     gathered per element as before (runs of Nq and Nq^2 contiguous doubles);
//   * the z rows, the row position, the neighbour rows and all per-thread index arithmetic are set up once per row;
//   * the packed SGS fluxes G and the LSRK residual are library-internal arrays and are stored ELEMENT-MAJOR,
//     [e][field][SLOT]: one bulk copy each per element instead of one per field (8 copies per element, not 24);
//     the residual is staged at the top of the iteration that consumes it;
//   * every asynchronous copy (bulk TMA and the cp.async gathers) is issued by a dedicated PRODUCER warp, so that the
//     ~20 issue cycles per bulk copy and the address arithmetic of the gathers never sit on the critical path of the
//     compute warps; the compute warps synchronise among themselves with a named barrier (twice per element), hand the
//     buffers of a finished element back to the producer with a non-blocking bar.arrive (only the producer waits), and
//     wait for data on mbarriers.
// The element-level phases (1: EOS + contravariant fluxes, 2: line tasks + face tasks, 3: assembly + fused LSRK update)
// and their arithmetic are those of cm_dg_kernels7.cuh; this file reuses its device functions.  P:L<n> = paper line.
#pragma once
#include "cm_dg_kernels7.cuh"

__device__ __forceinline__ void cm10_fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

template <int Nq, bool MOIST, int MODE> struct CmCfg10 {
  using C = CmCfg7<Nq, MOIST>;
  static constexpr int NF = C::NF, NV = C::NV, NTR = C::NTR, SLOT = C::SLOT, TS = C::TS_T;
  static constexpr int XS = (NTR * NF + 1) & ~1;                       // one xi trace / carry block [NTR][NF]
  static constexpr int OFF_Q = 0;                                      // [2][NV][SLOT]     state tiles (double-buffered)
  static constexpr int OFF_G = OFF_Q + 2 * NV * SLOT;                  // [2][2 NV][SLOT]   packed SGS fluxes land here; F^1, F^3 in place
  static constexpr int OFF_C = OFF_G + 4 * NV * SLOT;                  // [SLOT]            sound speed
  static constexpr int OFF_R = OFF_C + SLOT;                           // [NV][SLOT]        LSRK residual (MODE 1)
  static constexpr int OFF_F2 = OFF_R + (MODE == 1 ? NV * SLOT : 0);   // [NV][SLOT2]       F^2
  static constexpr int OFF_T = OFF_F2 + NV * C::SLOT2 + (NV * C::SLOT2 & 1);   // [NTB][4][TS]   eta / zeta neighbour traces, then rf
  static constexpr int TAILD = 3 * ((NTR * NF + 1) & ~1) + C::ZR * C::ZW + 6;   // xi blocks, z rows, mbarriers
  static constexpr size_t smem_with(int ntb) { return sizeof(double) * (size_t)(OFF_T + ntb * 4 * TS + TAILD); }
#ifndef CM_R_REGTHREADS
#define CM_R_REGTHREADS 512
#endif
  // resident CTAs the register budget allows (128 registers per thread at 512 threads per SM)
  static constexpr int REGCAP = C::cap(CM_R_REGTHREADS / (C::THREADS + 32), 16);
  // the trace buffer is double-buffered (gathers issued one element ahead) when that costs no resident CTA
  static constexpr int NTB = (C::cap(C::fit(smem_with(2)), REGCAP) == C::cap(C::fit(smem_with(1)), REGCAP)) ? 2 : 1;
  static constexpr int OFF_X = OFF_T + NTB * 4 * TS;                   // [3][XS]           xi- carry (x2), xi+ trace / rf
  static constexpr int OFF_Z = OFF_X + 3 * XS;                         // [ZR][ZW]          z rows
  static constexpr int OFF_M = OFF_Z + C::ZR * C::ZW;                  // mbarriers: tile buffer 0, 1, residual, gathered traces (x2), xi+ end trace
  static constexpr int DOUBLES = OFF_M + 6;
  static constexpr size_t SMEM = sizeof(double) * DOUBLES;
  static constexpr bool OK = SMEM <= 115712;                           // at least two CTAs per SM, else the cm7 kernels serve the order
  static constexpr int MINB = C::cap(C::fit(SMEM), REGCAP);
};

// position of the CTA's row in the tiled library order: grid = (PY * NSEG, Ez, (Ey/PY) * (Ex/L)), NSEG = L / S rows per
// x-chunk, blockIdx.x = eyl * NSEG + seg.  pos describes the row's FIRST element; its wallmask holds the eta / zeta bits.
struct Cm10Row { Cm7Pos pos; int S; bool wallL, wallR; int nbL, nbR, nb2, nb3, nb4, nb5; };

__device__ __forceinline__ Cm10Row cm10_row(const CmKP& p) {
  Cm10Row r;
  const int S = p.gS, NSEG = p.gL / S;
  const int bx = blockIdx.x, bz = blockIdx.z;
  Cm7Pos& q = r.pos;
  q.eyl = bx / NSEG; const int seg = bx - q.eyl * NSEG;
  q.yp = bz / p.gNXC; q.xc = bz - q.yp * p.gNXC;
  q.ez = blockIdx.y;
  q.exl = seg * S;
  q.e = (bz * p.gEz + q.ez) * (p.gPY * p.gL) + q.eyl * p.gL + q.exl;
  int m = 0;
  if (p.gbc[1]) { if (q.yp == 0 && q.eyl == 0) m |= 4; if (q.yp == p.gNYP - 1 && q.eyl == p.gPY - 1) m |= 8; }
  if (p.gbc[2]) { if (q.ez == 0) m |= 16; if (q.ez == p.gEz - 1) m |= 32; }
  q.wallmask = m;
  r.S = S;
  r.wallL = p.gbc[0] && q.xc == 0 && q.exl == 0;
  r.wallR = p.gbc[0] && q.xc == p.gNXC - 1 && q.exl + S == p.gL;
  r.nbL = cm7_neighbour(p, q, 0, 0);
  Cm7Pos last = q; last.exl = q.exl + S - 1;
  r.nbR = cm7_neighbour(p, last, 0, 1);
  r.nb2 = cm7_neighbour(p, q, 1, 0); r.nb3 = cm7_neighbour(p, q, 1, 1);   // the neighbour rows run parallel: + it
  r.nb4 = cm7_neighbour(p, q, 2, 0); r.nb5 = cm7_neighbour(p, q, 2, 1);
  return r;
}

// z rows of the row's elements (facing row below, own Nq rows, facing row above) to shared memory (producer warp)
template <int Nq>
__device__ __forceinline__ void cm10_zrows(const CmKP& p, const Cm7Pos& q, int lane, double* __restrict__ zt) {
  constexpr int ZR = Nq + 2;
  for (int c = lane; c < ZR * 7; c += 32) {
    const int r = c / 7, col = c - 7 * r;
    int row = q.ez * Nq + r - 1;
    if (r == 0) row = (q.wallmask & 16) ? -1 : (q.ez > 0 ? row : p.gEz * Nq - 1);
    if (r == ZR - 1) row = (q.wallmask & 32) ? -1 : (q.ez < p.gEz - 1 ? row : 0);
    if (row >= 0) cm7_cp8(zt + r * CM_ZSM_W + col, p.ztab + (size_t)row * CM_ZTAB_W + col);
  }
}

// One gather task of a producer lane: the neighbour trace of one eta / zeta face node (all NV + NGD values), or of one
// xi face node at the two ends of the row.  Fixed for the whole sweep: only the neighbour element advances with `it`.
struct Cm10Task { int f; int nb0; int np_; int goff; unsigned dst; };   // goff: first SGS value of direction d inside G[e]

template <int Nq, bool MOIST>
__device__ __forceinline__ Cm10Task cm10_task(const Cm10Row& r, int fn, const double* T, const double* X, int TS, int XS) {
  constexpr int NF = Nq * Nq;
  Cm10Task k;
  int f, m, d, s, nm, np_, kline;
  cm7_face_node<Nq>(fn, f, m, d, s, nm, np_, kline);
  k.f = (fn < 6 * NF) ? f : -1;
  k.np_ = np_;
  k.nb0 = (f == 0) ? r.nbL : (f == 1) ? r.nbR : (f == 2) ? r.nb2 : (f == 3) ? r.nb3 : (f == 4) ? r.nb4 : r.nb5;
  k.goff = d;
  k.dst = cm7_saddr((f < 2) ? X + 2 * XS * f + m : T + (f - 2) * TS + m);   // xi- trace (first element only) -> X[0], xi+ (last element) -> X[2]
  return k;
}

// issue the copies of one task for element `it` (Q field-major, G element-major [e][NG][SLOT])
// WHICH: 0 the eta / zeta faces of element it (+ the xi- face when it == 0) | 1 the xi+ face of the last element
template <int Nq, bool MOIST, int NV, int NG, int NGD, int SLOT, int WHICH>
__device__ __forceinline__ void cm10_task_issue(const CmKP& p, const Cm10Task& k, int it, int wm, unsigned tbuf_bytes) {
  constexpr int NF = Nq * Nq, NP = NF * Nq;
  if (k.f < 0 || ((wm >> k.f) & 1)) return;
  int nb = k.nb0;
  unsigned dst = k.dst;
  if (WHICH == 1) { if (k.f != 1) return; }
  else if (k.f == 1) return;
  else if (k.f == 0) { if (it != 0) return; }
  else { nb += it; dst += tbuf_bytes; }
  const double* src = p.Q + (size_t)nb * NP + k.np_;
#pragma unroll
  for (int v = 0; v < NV; ++v) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
    src += p.stride; dst += NF * 8;
  }
  if (NGD > 0) {
    const double* g = p.G + (size_t)nb * (NG * SLOT) + k.np_;
#pragma unroll
    for (int q = 0; q < NGD; ++q) {
      // index of the q-th value direction d needs in the packed SGS array (cm7_gidx), d = k.goff
      const int gi = (q == 3) ? 6 + k.goff : (q == 4) ? 9 + k.goff : (q == k.goff) ? k.goff : q + k.goff + 2;
      asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(g + gi * SLOT) : "memory");
      dst += NF * 8;
    }
  }
}

__device__ __forceinline__ void cm10_cp_arrive(uint64_t* bar) {   // arrive on bar once this thread's cp.async copies have landed
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(cm7_saddr(bar)) : "memory");
}
__device__ __forceinline__ void cm10_bar_compute(int nthreads) {   // barrier among the compute warps only (id 1)
  asm volatile("bar.sync 1, %0;" ::"r"(nthreads) : "memory");
}
// "buffers free" hand-over (id 2): the compute warps only ARRIVE (they never wait for the producer's instruction stream,
// only for its data), the producer warp waits until every compute thread has arrived
__device__ __forceinline__ void cm10_bar_release(int nthreads) { asm volatile("bar.arrive 2, %0;" ::"r"(nthreads) : "memory"); }
__device__ __forceinline__ void cm10_bar_acquire(int nthreads) { asm volatile("bar.sync 2, %0;" ::"r"(nthreads) : "memory"); }

// lifted numerical-flux part of one face node from the two states (cm7_tend_face with the operands in registers):
//   rf[v] = -(1/2) sJ n.F^+[v] - (1/2) sJ lambda (Y^-[v] - Y^+[v])          interior / periodic (eq. 27 with R1, R2, R6)
//   rf    = [0; -(p' + rho u_n (u_n + lambda)) sJ n; 0; 0] (+ sJ SHF on the bottom wall)   free-slip wall (A6-A7, R10)
template <int Nq, bool MOIST, bool SGS>
__device__ __forceinline__ void cm10_face_flux(const CmKP& p, const double (&Ym)[6], double cm_, const double (&Yp)[6],
                                               const double (&gp)[5], const double* __restrict__ zt, bool wall, int f, int d,
                                               int s, int kline, const double* __restrict__ qint, double (&rf)[6]) {
  using C = CmCfg7<Nq, MOIST>;
  constexpr int NV = C::NV;
  const double sgn = s ? 1.0 : -1.0;
  const double sJ = (d == 0) ? p.cA[0] : (d == 1) ? p.cA[1] : p.cA[2];
  const double A = sgn * sJ;
  const double mn = (d == 0) ? Ym[1] : (d == 1) ? Ym[2] : Ym[3];
  const double unm = sgn * (mn * cm_rcp(Ym[0]));                            // u^- . n
  CmSite st; CmPrim P;
  if (!wall) {
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
    if (f == 4) {                                                          // prescribed surface fluxes, drag law (App. A1);
      const double Aw[3] = {0.0, 0.0, -sJ};                                // qint: the node above the wall node in the own tile
      cm_surface_flux<MOIST>(p, Aw, sJ, Ym[0], qint, CmCfg7<Nq, MOIST>::SLOT, rf);
    }
  }
}

// MODE: 0 dQ := rhs | 1 LSRK stage reading the residual | 2 LSRK stage with A_s = 0 (residual not read)
// CTA = the compute warps (one thread per node, C::THREADS) + ONE producer warp that issues every asynchronous copy.
template <int Nq, bool MOIST, bool SGS, int MODE>
__global__ void __launch_bounds__(CmCfg7<Nq, MOIST>::THREADS + 32, CmCfg10<Nq, MOIST, MODE>::MINB) cm10_tendency_kernel(const __grid_constant__ CmKP p) {
  using C = CmCfg7<Nq, MOIST>;
  using R = CmCfg10<Nq, MOIST, MODE>;
  constexpr int NF = C::NF, NP = C::NP, N = Nq - 1, NV = C::NV, NG = C::NG, NGD = SGS ? C::NGD : 0, SLOT = C::SLOT, NFP = C::NFP;
  constexpr int THREADS = C::THREADS, TS = R::TS, XS = R::XS;
  extern __shared__ __align__(128) double smem10[];
  double* Qb = smem10 + R::OFF_Q;
  double* Gb = smem10 + R::OFF_G;
  double* ct = smem10 + R::OFF_C;
  double* Rt = smem10 + R::OFF_R;
  double* F2 = smem10 + R::OFF_F2;
  double* T = smem10 + R::OFF_T;
  double* X = smem10 + R::OFF_X;                      // X[0], X[1]: xi- carry of even / odd iterations; X[2]: xi+ trace / rf
  double* zt = smem10 + R::OFF_Z;
  uint64_t* mbar = reinterpret_cast<uint64_t*>(smem10 + R::OFF_M);   // [0], [1] tile buffers; [2] residual; [3], [4] gathered traces (even / odd element); [5] xi+ end trace

  const int t = threadIdx.x;
  const Cm10Row row = cm10_row(p);
  const int S = row.S;

  if (t == 0) {
    cm7_mbar_init(mbar, 1); cm7_mbar_init(mbar + 1, 1); cm7_mbar_init(mbar + 2, 1); cm7_mbar_init(mbar + 3, 32); cm7_mbar_init(mbar + 4, 32); cm7_mbar_init(mbar + 5, 32);
    cm7_fence_mbar_init();
  }
  __syncthreads();

  if (t >= THREADS) {
    // ================================================================ producer warp
    const int lane = t - THREADS;
    // bulk copies of the tiles of row element j into tile buffer bf (Q: one copy per field; G: element-major, one copy);
    // of its residual (element-major, one copy)
    auto issue_tile = [&](int j, int bf) {
      const int e = row.pos.e + j;
      const long long src = (long long)e * NP - (C::ODD ? (e & 1) : 0);
      const uint32_t mb = cm7_saddr(mbar + bf);
      cm7_mbar_expect_tx(mbar + bf, (uint32_t)((NV + (SGS ? NG : 0)) * SLOT * sizeof(double)));
      const double* g = p.Q + src; uint32_t d = cm7_saddr(Qb + bf * NV * SLOT);
#pragma unroll
      for (int v = 0; v < NV; ++v) { cm7_bulk_g2s_raw(d, g, SLOT * 8, mb); g += p.stride; d += SLOT * 8; }
      if (SGS) cm7_bulk_g2s_raw(cm7_saddr(Gb + bf * 2 * NV * SLOT), p.G + (size_t)e * (NG * SLOT), NG * SLOT * 8, mb);
    };
    auto issue_res = [&](int j) {
      const int e = row.pos.e + j;
      cm7_mbar_expect_tx(mbar + 2, (uint32_t)(NV * SLOT * sizeof(double)));
      cm7_bulk_g2s_raw(cm7_saddr(Rt), p.dQ + (size_t)e * (NV * SLOT), NV * SLOT * 8, cm7_saddr(mbar + 2));
    };
    if (lane == 0) issue_tile(0, 0);
    cm10_zrows<Nq>(p, row.pos, lane, zt);
    constexpr int NTASK = (6 * NF + 31) / 32;
    Cm10Task task[NTASK];
#pragma unroll
    for (int q = 0; q < NTASK; ++q) task[q] = cm10_task<Nq, MOIST>(row, lane + 32 * q, T, X, TS, XS);
    auto wall_mask = [&](int j) { return row.pos.wallmask | ((j == 0 && row.wallL) ? 1 : 0) | ((j == S - 1 && row.wallR) ? 2 : 0); };
    auto gather = [&](int j) {                        // eta / zeta traces of element j into trace buffer j % NTB
      const int wm = wall_mask(j);
      const unsigned tb = (unsigned)((j % R::NTB) * 4 * TS * sizeof(double));
#pragma unroll
      for (int q = 0; q < NTASK; ++q) cm10_task_issue<Nq, MOIST, NV, NG, NGD, SLOT, 0>(p, task[q], j, wm, tb);
      cm10_cp_arrive(mbar + 3 + (j & 1));             // one mbarrier per parity of j: arrivals of consecutive elements never mix
    };
    if (R::NTB == 2) gather(0);
    for (int j = 0; j < S; ++j) {
      cm10_bar_acquire(THREADS + 32);                  // the compute warps are done with every buffer of element j-1
      if (lane == 0) {
        cm10_fence_proxy_async();                      // generic-proxy accesses of the buffers before the async-proxy writes
        if (j + 1 < S) issue_tile(j + 1, (j + 1) & 1);
        if (MODE == 1) issue_res(j);
      }
      __syncwarp();
      if (R::NTB == 2) { if (j + 1 < S) gather(j + 1); } else gather(j);
      if (j == S - 1) {                                // xi+ trace of the last element of the row
        const int wm = wall_mask(j);
#pragma unroll
        for (int q = 0; q < NTASK; ++q) cm10_task_issue<Nq, MOIST, NV, NG, NGD, SLOT, 1>(p, task[q], j, wm, 0u);
        cm10_cp_arrive(mbar + 5);
      }
      if (j + 2 < S) {
        // pull what the next step will copy into L2 (tile j+2, residual j+1), so that its bulk copies hit L2
        const int e = row.pos.e + j + 2;
        if (lane < NV) cm7_prefetch_l2(p.Q + (size_t)lane * p.stride + ((long long)e * NP - (C::ODD ? (e & 1) : 0)), SLOT * 8);
        else if (SGS && lane == NV) cm7_prefetch_l2(p.G + (size_t)e * (NG * SLOT), NG * SLOT * 8);
        else if (MODE == 1 && lane == NV + 1) cm7_prefetch_l2(p.dQ + (size_t)(e - 1) * (NV * SLOT), NV * SLOT * 8);
      }
      __syncwarp();
    }
    return;
  }

  // ================================================================== compute warps
  const int n = t;
  const bool node = t < NP;
  const int k_ = n / NF, j_ = (n - k_ * NF) / Nq, i_ = n - k_ * NF - j_ * Nq;
  const int n2 = n + (C::PS2 - NF) * k_;               // index in the F^2 tiles
  CmSite st;
  if (node) {
    const double2* zr = reinterpret_cast<const double2*>(p.ztab + (size_t)(row.pos.ez * Nq + k_) * CM_ZTAB_W);
    const double2 a = __ldg(zr), b = __ldg(zr + 1), c = __ldg(zr + 2), d = __ldg(zr + 3);
    st.Phi = a.x; st.rho_r = a.y; st.rhoe_r = b.x; st.rhoq_r = b.y; st.E_r = c.x; st.q_r = c.y; st.icvm_r = d.x; st.taus = d.y;
  }

  for (int it = 0; it < S; ++it) {
    const int b = it & 1;
    const int e = row.pos.e + it;
    const int sh = C::ODD ? (e & 1) : 0;
    const int wm = row.pos.wallmask | ((it == 0 && row.wallL) ? 1 : 0) | ((it == S - 1 && row.wallR) ? 2 : 0);
    const bool more = it + 1 < S;
    // releases the buffers of the previous iteration to the producer WITHOUT waiting: a warp that has finished phase 3
    // starts phase 1 of the next element at once.  What phase 1 writes is either private to the thread's own node (F^2,
    // c) or lies in the other tile buffer; the xi- carry is written behind the first compute barrier for this reason.
    // Every compute thread orders its own generic-proxy stores to the buffers (F^1 / F^3 over G, the xi carry, the face
    // results) before the async-proxy bulk copies that will overwrite them: the PTX memory model makes a proxy fence
    // cover only the executing thread's prior accesses, so the fence must run in the writers before they signal the
    // producer (the pattern of a TMA-store fence), not only in the producer after the barrier.
    cm10_fence_proxy_async();
    cm10_bar_release(THREADS + 32);
    cm7_mbar_wait(mbar + b, (it >> 1) & 1);

    double* Qs = Qb + b * NV * SLOT + sh; double* Fs = Gb + b * 2 * NV * SLOT; double* cs = ct;   // G is element-major: no shift
    // ---- phase 1: primitives and contravariant fluxes of the own node (F^1, F^3 overwrite G in place)
    double buoy = 0.0;
    double Y[6], gc[5];
    if (node) {
      double g[12]; CmPrim P;
#pragma unroll
      for (int v = 0; v < NV; ++v) Y[v] = Qs[v * SLOT + n];
      if (SGS) {
#pragma unroll
        for (int k = 0; k < NG; ++k) g[k] = Fs[k * SLOT + n];
#pragma unroll
        for (int k = 0; k < NGD; ++k) gc[k] = g[cm7_gidx(0, k)];
      }
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
    cm10_bar_compute(THREADS);
    if (node && i_ == N && more) {                     // the i = N plane is the xi- trace of the next element (every warp
      double* xl = X + (b ^ 1) * XS + (j_ + Nq * k_);  // has left phase 3 of the previous element, which read this block)
#pragma unroll
      for (int v = 0; v < NV; ++v) xl[v * NF] = Y[v];
      if (SGS)
#pragma unroll
        for (int k = 0; k < NGD; ++k) xl[(NV + k) * NF] = gc[k];
    }

    // ---- phase 2: line tasks, then face tasks
    for (int lt = t; lt < 3 * NFP; lt += THREADS) {
      const int d = lt / NFP, l = lt % NFP;
      if (d == 0) { if (l < NF) cm7_tend_line<Nq, NV, SLOT, 1, 0>(p, Fs + Nq * l, wm); }
      else if (d == 1) { int base; if (cm7_yline<Nq>(l, base)) cm7_tend_line<Nq, NV, C::SLOT2, Nq, 1>(p, F2 + base, wm); }
      else { if (l < NF) cm7_tend_line<Nq, NV, SLOT, NF, 2>(p, Fs + NV * SLOT + l, wm); }
    }
    cm7_mbar_wait(mbar + 3 + b, (it >> 1) & 1);        // gathered traces (and, first iteration, the z rows) have landed
    if (!more) cm7_mbar_wait(mbar + 5, 0);             // last element: the gathered xi+ trace
    double* Tb = T + (it % R::NTB) * 4 * TS;
    if (more) cm7_mbar_wait(mbar + (b ^ 1), ((it + 1) >> 1) & 1);   // the next tile (xi+ faces read its i = 0 plane)
    const int shn = C::ODD ? ((e + 1) & 1) : 0;
    for (int fn = THREADS - 1 - t; fn < 6 * NF; fn += THREADS) {
      int f, m, d, s, nm, np_, kline;
      cm7_face_node<Nq>(fn, f, m, d, s, nm, np_, kline);
      const bool wall = (wm >> f) & 1;
      double Ym[6], Yp[6], gp[5], rf[6];
#pragma unroll
      for (int v = 0; v < NV; ++v) Ym[v] = Qs[v * SLOT + nm];
      const double cm_ = cs[nm];
      double* out;
      if (f == 1 && more) {                            // xi+ inside the row: the neighbour's tile is in the other buffer
        out = X + 2 * XS + m;
        const double* qn = Qb + (b ^ 1) * NV * SLOT + shn + np_;
        const double* gn = Gb + (b ^ 1) * 2 * NV * SLOT + np_;
#pragma unroll
        for (int v = 0; v < NV; ++v) Yp[v] = qn[v * SLOT];
        if (SGS)
#pragma unroll
          for (int k = 0; k < NGD; ++k) gp[k] = gn[cm7_gidx(0, k) * SLOT];
      } else {
        out = (f == 0) ? X + b * XS + m : (f == 1) ? X + 2 * XS + m : Tb + (f - 2) * TS + m;
        if (!wall) {
#pragma unroll
          for (int v = 0; v < NV; ++v) Yp[v] = out[v * NF];
          if (SGS)
#pragma unroll
            for (int k = 0; k < NGD; ++k) gp[k] = out[(NV + k) * NF];
        }
      }
      cm10_face_flux<Nq, MOIST, SGS>(p, Ym, cm_, Yp, gp, zt, wall, f, d, s, kline, Qs + nm + NF, rf);
#pragma unroll
      for (int v = 0; v < NV; ++v) out[v * NF] = rf[v];
    }
    if (MODE == 1) cm7_mbar_wait(mbar + 2, it & 1);    // residual tile (issued at the top of this iteration)
    cm10_bar_compute(THREADS);

    // ---- phase 3: assemble the tendency of the own node and update
    if (node) {
      const double* Rs = Rt;                           // residual: element-major [e][NV][SLOT] (MODE 1, 2)
      double acc[6], lift[6], Ro[6];
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        acc[v] = Fs[v * SLOT + n] + F2[v * C::SLOT2 + n2] + Fs[(NV + v) * SLOT + n];
        lift[v] = 0.0;
        if (MODE == 1) Ro[v] = Rs[v * SLOT + n];
      }
      const int c3[3] = {i_, j_, k_};
      const int m3[3] = {j_ + Nq * k_, i_ + Nq * k_, i_ + Nq * j_};
      double lf[3][6];                                 // rf of the up to three faces through the node: independent
#pragma unroll                                         // (predicated) loads, all in flight together
      for (int d = 0; d < 3; ++d) {
        const bool on = c3[d] == 0 || c3[d] == N, hi = c3[d] == N;
        const double* tr = (d == 0) ? (hi ? X + 2 * XS : X + b * XS) : T + (it % R::NTB) * 4 * TS + (2 * d - 2 + (hi ? 1 : 0)) * TS;
        tr += m3[d];
#pragma unroll
        for (int v = 0; v < NV; ++v) lf[d][v] = on ? tr[v * NF] : 0.0;
      }
#pragma unroll
      for (int v = 0; v < NV; ++v) lift[v] = (lf[0][v] + lf[1][v]) + lf[2][v];
      const size_t idx = (size_t)e * NP + n;
      double* o1 = (MODE == 0) ? p.dQ + idx : p.dQ + (size_t)e * (NV * SLOT) + n;
      const long long s1 = (MODE == 0) ? p.stride : (long long)SLOT;
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
          __stcs(o2, Y[v] + p.rkb * dnew);
          o2 += p.stride;
        }
        o1 += s1;
      }
    }
  }
}

