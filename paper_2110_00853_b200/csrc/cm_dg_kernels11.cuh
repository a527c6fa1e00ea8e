// cm_dg_kernels11.cuh -- CTA-per-element tendency and gradient kernels for STORED-METRIC meshes (geom != 0: terrain-
// following and fully warped bricks, per-node reference state): the decomposition of the flat CTA-per-element kernels
// (cm_dg_kernels7.cuh) with the geometry as data.
//
// Why (profiles/r2_stored_metric.md): the thread-per-node kernel of cm_dg_kernels2.cuh waits on global loads at the start of
// every phase (ncu: 38 % of its warp time in long-scoreboard stalls, 20 % at barriers, 0.43 eligible warps per scheduler).
// Here everything the element needs arrives asynchronously at CTA start, exactly as on flat meshes:
//   * the launch grid is the tiled element order, so the element's position, its neighbours and its wall flags follow from
//     blockIdx (no connectivity load in front of the data loads);
//   * one elected thread fetches the element's own tiles by 1-D bulk TMA behind an mbarrier: Q (NV), packed SGS fluxes G
//     (NG, field-major as the stored-metric gradient kernel writes them), LSRK residual (NV), and the per-node geometry
//     the tendency needs -- Ja (9), 1/J, z, tau_s -- plus the reference state (rho_r, rhoe_r, [rhoq_r]);
//   * every thread copies the neighbour traces of its face node(s) with 8-byte cp.async: Q (NV), all NG packed SGS values
//     (the face normal is not axis-aligned), z and the reference state of the neighbour's coincident node;
//   * phase 1 (thread per node): EOS, contravariant fluxes Ja^d . (F1 + F2) (eq. 24, 32) -- F^1, F^3 in place of G, F^2 in
//     its own tiles; phase 2: line tasks (cm7_tend_line: D_d F^d in place + the own-side half of the face term, which is
//     the contravariant flux itself) and face tasks (Rusanov with A = +-Ja^d of the own face node, central SGS flux, mirror
//     walls, surface fluxes); phase 3: 1/J, gravity, sponge, fused LSRK update.
// Arithmetic follows cm_dg_physics.cuh and is the one of cm2_tendency_kernel.  P:L<n> = paper line.
#pragma once
#include "cm_dg_kernels7.cuh"

// TERR: terrain-following mesh (geom == 1: x and y stay a uniform brick, only z is warped).  Then
//   Ja^1 = (h_y/2 z_zeta, 0, 0),  Ja^2 = (0, h_x/2 z_zeta, 0),  Ja^3 = (-h_y/2 z_xi, -h_x/2 z_eta, h_x h_y/4)      (eq. 24)
// and three of the nine metric tiles carry everything: Ja[0], Ja[6], Ja[7] (Ja[4] = Ja[0] h_x/h_y, Ja[8] is a constant).
template <bool TERR> struct Cm11Geo {
  static constexpr int NGEO = TERR ? 6 : 12;            // tiles: Ja (9 | 3), 1/J, z, tau_s
  static constexpr int S_INVJ = NGEO - 3, S_Z = NGEO - 2, S_TAUS = NGEO - 1;
  __host__ __device__ static constexpr int field(int k) {   // tile k of the geometry block -> CmKP::geo field
    return TERR ? (k == 0 ? 0 : k == 1 ? 6 : k == 2 ? 7 : k == 3 ? 9 : k == 4 ? 10 : 15) : (k < 11 ? k : 15);
  }
  // metric entry Ja[m] (m = 3 d + c, compile-time in unrolled code) of node n; r = h_x / h_y, a3 = h_x h_y / 4
  template <int SLOT>
  __device__ __forceinline__ static double ja(const double* __restrict__ geo, int m, int n, double r, double a3) {
    if (!TERR) return geo[m * SLOT + n];
    return (m == 0) ? geo[n] : (m == 4) ? geo[n] * r : (m == 6) ? geo[SLOT + n] : (m == 7) ? geo[2 * SLOT + n] : (m == 8) ? a3 : 0.0;
  }
};

template <int Nq, bool MOIST, bool SGS, int MODE, bool TERR = false> struct CmCfg11 {
  using C = CmCfg7<Nq, MOIST>;
  static constexpr int NF = C::NF, NP = C::NP, NV = C::NV, NG = SGS ? C::NG : 0, SLOT = C::SLOT, THREADS = C::THREADS;
  static constexpr int NGEO = Cm11Geo<TERR>::NGEO;      // fields 0..8, 9, 10, 15 of CmKP::geo, or 0, 6, 7, 9, 10, 15
  static constexpr int NREF = MOIST ? 3 : 2;            // rho_r, rhoe_r, [rhoq_r]
  static constexpr int NTR = NV + NG + 1 + NREF;        // trace values per face node: state, SGS fluxes, z, reference
  static constexpr int TS = C::fstride(NTR);
  static constexpr int OFF_Q = 0;                                        // [NV][SLOT]
  static constexpr int OFF_F = OFF_Q + NV * SLOT;                        // [2 NV][SLOT]  G lands here; F^1, F^3 in place
  static constexpr int OFF_C = OFF_F + 2 * NV * SLOT;                    // [SLOT]        sound speed
  static constexpr int OFF_R = OFF_C + SLOT;                             // [NV][SLOT]    LSRK residual (MODE 1)
  static constexpr int OFF_F2 = OFF_R + (MODE == 1 ? NV * SLOT : 0);     // [NV][SLOT2]   F^2
  static constexpr int OFF_GEO = OFF_F2 + NV * C::SLOT2 + (NV * C::SLOT2 & 1);   // [NGEO][SLOT]
  static constexpr int OFF_REF = OFF_GEO + NGEO * SLOT;                  // [NREF][SLOT]
  static constexpr int OFF_T = OFF_REF + NREF * SLOT;                    // [6][TS]       traces, then rf
  static constexpr int OFF_M = OFF_T + 5 * TS + NTR * NF + (NTR * NF & 1);
  static constexpr int DOUBLES = OFF_M + 2;
  static constexpr size_t SMEM = sizeof(double) * DOUBLES;
  static constexpr bool OK = SMEM <= 115712;                             // at least two CTAs per SM, else cm2 serves the order
  static constexpr int MINB = C::cap(C::fit(SMEM), C::cap(640 / THREADS, 16));
};

// face task on a stored-metric mesh: replaces the trace of face node fn by
//   rf[v] = -(1/2) A.F^+[v] - (1/2) sJ lambda (Y^-[v] - Y^+[v])     interior / periodic (eq. 27 with R1, R2; P:L274 with R6)
//   rf    = [0; -(p' + rho u_n (u_n + lambda)) A; 0; 0] + surface fluxes on the bottom wall      free-slip wall (A6-A7, R10)
// with A = +-Ja^d of the own face node (outward, |A| = sJ)
template <int Nq, bool MOIST, bool SGS, int MODE, bool TERR>
__device__ __forceinline__ void cm11_tend_face(const CmKP& p, const double* __restrict__ Qs, const double* __restrict__ cs,
                                               const double* __restrict__ geo, const double* __restrict__ ref, double* __restrict__ T,
                                               int wallmask, int fn) {
  using R = CmCfg11<Nq, MOIST, SGS, MODE, TERR>;
  using GG = Cm11Geo<TERR>;
  constexpr int NF = R::NF, NV = R::NV, NG = R::NG, SLOT = R::SLOT, TS = R::TS, NREF = R::NREF;
  int f, m, d, s, nm, np_, kline;
  cm7_face_node<Nq>(fn, f, m, d, s, nm, np_, kline);
  const bool wall = (wallmask >> f) & 1;
  double* tr = T + f * TS + m;
  const double sgn = s ? 1.0 : -1.0;
  double A[3];
  if (TERR) {
    const double r = p.cA[1] * cm_rcp(p.cA[0]), a0 = geo[nm];
    A[0] = sgn * ((d == 0) ? a0 : (d == 1) ? 0.0 : geo[SLOT + nm]);
    A[1] = sgn * ((d == 0) ? 0.0 : (d == 1) ? a0 * r : geo[2 * SLOT + nm]);
    A[2] = sgn * ((d == 2) ? p.cA[2] : 0.0);
  } else {
#pragma unroll
    for (int c = 0; c < 3; ++c) A[c] = sgn * geo[(3 * d + c) * SLOT + nm];
  }
  const double sJ = cm_sqrt(A[0] * A[0] + A[1] * A[1] + A[2] * A[2]);
  double Ym[6];
#pragma unroll
  for (int v = 0; v < NV; ++v) Ym[v] = Qs[v * SLOT + nm];
  const double cm_ = cs[nm];
  const double uAm = (Ym[1] * A[0] + Ym[2] * A[1] + Ym[3] * A[2]) * cm_rcp(Ym[0]);      // sJ (u^- . n)
  double rf[6];
  CmSite st; CmPrim P;
  if (!wall) {
    double Yp[6], gp[12];
#pragma unroll
    for (int v = 0; v < NV; ++v) Yp[v] = tr[v * NF];
    if (SGS)
#pragma unroll
      for (int k = 0; k < NG; ++k) gp[k] = tr[(NV + k) * NF];
    st.Phi = p.th.grav * tr[(NV + NG) * NF]; st.taus = 0.0;
    if (p.use_ref) {
      st.rho_r = tr[(NV + NG + 1) * NF]; st.rhoe_r = tr[(NV + NG + 2) * NF];
      st.rhoq_r = MOIST ? tr[(NV + NG + NREF) * NF] : 0.0;
      st.q_r = MOIST ? st.rhoq_r * cm_rcp(st.rho_r) : 0.0;
      st.icvm_r = MOIST ? cm_rcp(p.th.c_vd + p.th.b * st.q_r) : p.th.icvd;
      st.E_r = st.rhoe_r - st.rho_r * st.Phi - st.rhoq_r * p.th.I_v0;
    } else { st.rho_r = st.rhoe_r = st.rhoq_r = st.E_r = st.q_r = 0.0; st.icvm_r = 0.0; }
    cm_eos<MOIST>(p, Yp, st, P);
    double Fp[6];
    cm_flux_dir<MOIST>(Yp, P, SGS, gp, A[0], A[1], A[2], Fp);
    const double uAp = A[0] * P.u + A[1] * P.v + A[2] * P.w;
    const double lamsJ = fmax(fabs(uAm) + cm_ * sJ, fabs(uAp) + cm_sqrt(P.c2) * sJ);   // sJ lambda (R2)
#pragma unroll
    for (int v = 0; v < NV; ++v) rf[v] = -0.5 * Fp[v] - 0.5 * lamsJ * (Ym[v] - Yp[v]);
  } else {
    st.Phi = p.th.grav * geo[GG::S_Z * SLOT + nm]; st.taus = 0.0;
    if (p.use_ref) {
      st.rho_r = ref[nm]; st.rhoe_r = ref[SLOT + nm];
      st.rhoq_r = MOIST ? ref[2 * SLOT + nm] : 0.0;
      st.q_r = MOIST ? st.rhoq_r * cm_rcp(st.rho_r) : 0.0;
      st.icvm_r = MOIST ? cm_rcp(p.th.c_vd + p.th.b * st.q_r) : p.th.icvd;
      st.E_r = st.rhoe_r - st.rho_r * st.Phi - st.rhoq_r * p.th.I_v0;
    } else { st.rho_r = st.rhoe_r = st.rhoq_r = st.E_r = st.q_r = 0.0; st.icvm_r = 0.0; }
    cm_eos<MOIST>(p, Ym, st, P);
    const double un = uAm * cm_rcp(sJ);
    const double lam = fabs(un) + cm_;
    const double mom = -(P.pp + Ym[0] * un * (un + lam));
#pragma unroll
    for (int v = 0; v < NV; ++v) rf[v] = 0.0;
    rf[1] = mom * A[0]; rf[2] = mom * A[1]; rf[3] = mom * A[2];
    if (f == 4) cm_surface_flux<MOIST>(p, A, sJ, Ym[0], Qs + nm + NF, SLOT, rf);   // the node above nm: first interior layer
  }
#pragma unroll
  for (int v = 0; v < NV; ++v) tr[v * NF] = rf[v];
}

// MODE: 0 dQ := rhs | 1 LSRK stage reading the residual | 2 LSRK stage with A_s = 0 (residual not read)
template <int Nq, bool MOIST, bool SGS, int MODE, bool TERR>
__global__ void __launch_bounds__(CmCfg7<Nq, MOIST>::THREADS, CmCfg11<Nq, MOIST, SGS, MODE, TERR>::MINB) cm11_tendency_kernel(const __grid_constant__ CmKP p) {
  using C = CmCfg7<Nq, MOIST>;
  using R = CmCfg11<Nq, MOIST, SGS, MODE, TERR>;
  using GG = Cm11Geo<TERR>;
  constexpr int NF = C::NF, NP = C::NP, N = Nq - 1, NV = C::NV, NG = R::NG, SLOT = C::SLOT, NFP = C::NFP, THREADS = C::THREADS;
  constexpr int TS = R::TS, NREF = R::NREF, NGEO = R::NGEO;
  extern __shared__ __align__(128) double smem11[];
  double* Qt = smem11 + R::OFF_Q;
  double* Ft = smem11 + R::OFF_F;
  double* ct = smem11 + R::OFF_C;
  double* Rt = smem11 + R::OFF_R;
  double* F2 = smem11 + R::OFF_F2;
  double* Gt = smem11 + R::OFF_GEO;
  double* Ht = smem11 + R::OFF_REF;
  double* T = smem11 + R::OFF_T;
  uint64_t* mbar = reinterpret_cast<uint64_t*>(smem11 + R::OFF_M);

  const int t = threadIdx.x;
  const Cm7Pos pos = cm7_position(p);
  const int e = pos.e;
  const int sh = C::ODD ? (e & 1) : 0;
  const int nref = p.use_ref ? NREF : 0;

  if (t == THREADS - 32) { cm7_mbar_init(mbar, 1); cm7_fence_mbar_init(); }
  __syncthreads();
  if (t == THREADS - 32) {                             // lane 0 of the last warp issues the bulk copies of the own tiles
    const long long src = (long long)e * NP - sh;
    const uint32_t mb = cm7_saddr(mbar);
    cm7_mbar_expect_tx(mbar, (uint32_t)((NV + NG + (MODE == 1 ? NV : 0) + NGEO + nref) * SLOT * sizeof(double)));
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
    {
      uint32_t d = cm7_saddr(Gt);
#pragma unroll
      for (int k = 0; k < NGEO; ++k) { cm7_bulk_g2s_raw(d, p.geo + (size_t)GG::field(k) * p.stride + src, SLOT * 8, mb); d += SLOT * 8; }
    }
    {
      uint32_t d = cm7_saddr(Ht);
      for (int k = 0; k < nref; ++k) { cm7_bulk_g2s_raw(d, p.ref + (size_t)k * p.stride + src, SLOT * 8, mb); d += SLOT * 8; }
    }
  } else if (t > THREADS - 32 && p.ahead > 0 && e + p.ahead < p.Ne) {
    // the other lanes of that warp pull the tiles of the element one wave further on in the launch order into L2
    const int ea = e + p.ahead;
    const long long src = (long long)ea * NP - (C::ODD ? (ea & 1) : 0);
    const int ntile = NV + NG + (MODE == 1 ? NV : 0) + NGEO + nref;
    for (int j = t - (THREADS - 32) - 1; j < ntile; j += 31) {
      int k = j; const double* g;
      if (k < NV) g = p.Q + (size_t)k * p.stride;
      else if ((k -= NV) < NG) g = p.G + (size_t)k * p.stride;
      else if ((k -= NG) < (MODE == 1 ? NV : 0)) g = p.dQ + (size_t)k * p.stride;
      else if ((k -= (MODE == 1 ? NV : 0)) < NGEO) g = p.geo + (size_t)GG::field(k) * p.stride;
      else g = p.ref + (size_t)(k - NGEO) * p.stride;
      cm7_prefetch_l2(g + src, SLOT * 8);
    }
  }
  // neighbour traces (phase 2 needs them): the thread that will run the face task of node fn copies them
  for (int fn = THREADS - 1 - t; fn < 6 * NF; fn += THREADS) {
    int f, m, d, s, nm, np_, kline;
    cm7_face_node<Nq>(fn, f, m, d, s, nm, np_, kline);
    if (!((pos.wallmask >> f) & 1)) {
      const int nb = cm7_neighbour(p, pos, d, s);
      const size_t idp = (size_t)nb * NP + np_;
      double* dst = T + f * TS + m;
      const double* src = p.Q + idp;
#pragma unroll
      for (int v = 0; v < NV; ++v) { cm7_cp8(dst + v * NF, src); src += p.stride; }
      if (SGS) {
        const double* g = p.G + idp;
#pragma unroll
        for (int k = 0; k < NG; ++k) { cm7_cp8(dst + (NV + k) * NF, g); g += p.stride; }
      }
      cm7_cp8(dst + (NV + NG) * NF, p.geo + 10 * p.stride + idp);
      for (int k = 0; k < nref; ++k) cm7_cp8(dst + (NV + NG + 1 + k) * NF, p.ref + (size_t)k * p.stride + idp);
    }
  }
  cm7_cp_commit();

  double* Qs = Qt + sh; double* Fs = Ft + sh; double* cs = ct + sh; const double* Rs = Rt + sh;
  const double* geo = Gt + sh; const double* ref = Ht + sh;
  const int n = t;
  const bool node = t < NP;
  const int k_ = n / NF, j_ = (n - k_ * NF) / Nq, i_ = n - k_ * NF - j_ * Nq;
  const int n2 = n + (C::PS2 - NF) * k_;               // index in the F^2 tiles
  cm7_mbar_wait(mbar, 0);

  // ---- phase 1: primitives and contravariant fluxes of the own node (F^1, F^3 overwrite G in place)
  double buoy = 0.0, taus = 0.0, invJ = 0.0;
  double Y[6];
  if (node) {
    double g[12]; CmPrim P; CmSite st;
#pragma unroll
    for (int v = 0; v < NV; ++v) Y[v] = Qs[v * SLOT + n];
    if (SGS)
#pragma unroll
      for (int k = 0; k < NG; ++k) g[k] = Fs[k * SLOT + n];
    const double hr = TERR ? p.cA[1] * cm_rcp(p.cA[0]) : 0.0;
    double Ja[9];
#pragma unroll
    for (int m = 0; m < 9; ++m) Ja[m] = GG::template ja<SLOT>(geo, m, n, hr, p.cA[2]);
    invJ = geo[GG::S_INVJ * SLOT + n]; taus = geo[GG::S_TAUS * SLOT + n];
    st.Phi = p.th.grav * geo[GG::S_Z * SLOT + n]; st.taus = taus;
    if (p.use_ref) {
      st.rho_r = ref[n]; st.rhoe_r = ref[SLOT + n];
      st.rhoq_r = MOIST ? ref[2 * SLOT + n] : 0.0;
      st.q_r = MOIST ? st.rhoq_r * cm_rcp(st.rho_r) : 0.0;
      st.icvm_r = MOIST ? cm_rcp(p.th.c_vd + p.th.b * st.q_r) : p.th.icvd;
      st.E_r = st.rhoe_r - st.rho_r * st.Phi - st.rhoq_r * p.th.I_v0;
    } else { st.rho_r = st.rhoe_r = st.rhoq_r = st.E_r = st.q_r = 0.0; st.icvm_r = 0.0; }
    cm_eos<MOIST>(p, Y, st, P);
    buoy = P.drho * p.th.grav;
    cs[n] = cm_sqrt(P.c2);
    double Fa[6], Fb[6], Fc[6];
    if (TERR) {                                        // Ja^1, Ja^2 are axis-aligned
      cm_flux_axis<MOIST, 0>(Y, P, SGS, g, Ja[0], Fa);
      cm_flux_axis<MOIST, 1>(Y, P, SGS, g, Ja[4], Fb);
    } else {
      cm_flux_dir<MOIST>(Y, P, SGS, g, Ja[0], Ja[1], Ja[2], Fa);
      cm_flux_dir<MOIST>(Y, P, SGS, g, Ja[3], Ja[4], Ja[5], Fb);
    }
    cm_flux_dir<MOIST>(Y, P, SGS, g, Ja[6], Ja[7], Ja[8], Fc);
#pragma unroll
    for (int v = 0; v < NV; ++v) { Fs[v * SLOT + n] = Fa[v]; Fs[(NV + v) * SLOT + n] = Fc[v]; F2[v * C::SLOT2 + n2] = Fb[v]; }
  }
  __syncthreads();

  // ---- phase 2: line tasks (one warp per direction), then face tasks (handed out from the last thread downwards)
  for (int lt = t; lt < 3 * NFP; lt += THREADS) {
    const int d = lt / NFP, l = lt % NFP;
    if (d == 0) { if (l < NF) cm7_tend_line<Nq, NV, SLOT, 1, 0>(p, Fs + Nq * l, pos.wallmask); }
    else if (d == 1) { int base; if (cm7_yline<Nq>(l, base)) cm7_tend_line<Nq, NV, C::SLOT2, Nq, 1>(p, F2 + base, pos.wallmask); }
    else { if (l < NF) cm7_tend_line<Nq, NV, SLOT, NF, 2>(p, Fs + NV * SLOT + l, pos.wallmask); }
  }
  cm7_cp_wait_all();                                   // this thread's trace copies have landed
  for (int fn = THREADS - 1 - t; fn < 6 * NF; fn += THREADS) cm11_tend_face<Nq, MOIST, SGS, MODE, TERR>(p, Qs, cs, geo, ref, T, pos.wallmask, fn);
  __syncthreads();

  // ---- phase 3: assemble the tendency of the own node and update
  if (node) {
    double acc[6], Ro[6], lf[3][6];
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      acc[v] = Fs[v * SLOT + n] + F2[v * C::SLOT2 + n2] + Fs[(NV + v) * SLOT + n];
      if (MODE == 1) Ro[v] = Rs[v * SLOT + n];
    }
    const int c3[3] = {i_, j_, k_};
    const int m3[3] = {j_ + Nq * k_, i_ + Nq * k_, i_ + Nq * j_};
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const bool on = c3[d] == 0 || c3[d] == N;
      const double* tr = T + (2 * d + (c3[d] == N ? 1 : 0)) * TS + m3[d];
#pragma unroll
      for (int v = 0; v < NV; ++v) lf[d][v] = on ? tr[v * NF] : 0.0;
    }
    const size_t idx = (size_t)e * NP + n;
    double* o1 = p.dQ + idx;
    double* o2 = p.Qnew + idx;
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      const double lift = (lf[0][v] + lf[1][v]) + lf[2][v];
      double rhs = -invJ * (acc[v] - p.inv_w0 * lift);
      if (v == 3) rhs -= buoy;                                   // -(rho - rho_r) grad Phi   (eq. 4)
      if (v >= 1 && v <= 3) rhs -= taus * (Y[v] - Y[0] * p.urelax[v - 1]);   // Rayleigh sponge (A4); tau_s = 0 outside the layer
      if (MODE == 0) {
        __stcs(o1, rhs);
      } else {
        const double dnew = (MODE == 1) ? p.rka * Ro[v] + p.dt * rhs : p.dt * rhs;   // a5: dU <- A_s dU + dt RHS ; U <- U + B_s dU
        __stcs(o1, dnew);
        __stcs(o2, Y[v] + p.rkb * dnew);
        o2 += p.stride;
      }
      o1 += p.stride;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// a2 on stored-metric meshes: BR1 auxiliary gradient + eddy-viscosity closure, same staging as the tendency kernel above.
//   own tiles by bulk TMA: Q (NV) and the geometry fields 0..14 (Ja 9, 1/J, z, (C_s Delta)^2, Delta_m^2 3);
//   neighbour traces by cp.async: Q (NV) and z of the neighbour's node;
//   phase 1: gradient variables s = u, v, w, h_tot, [q_t], [theta_v] in place of the state (eq. 33, 35, 37, 40);
//   phase 2: face tasks  s* - s^- = (s^+ - s^-)/2 (eq. 30-31), wall: u* = u - (n.u) n with n from Ja^d (A6), scalars kept (A8);
//            line tasks  D_d s in reference space;
//   phase 3: lifted jumps, G = (1/J) sum_d Ja^d (D_d s + lift_d) (eq. 28-29 with eq. 24), closure, field-major store.
// RAW: the 15 raw gradients (cm_dg_gradient) | packed SGS fluxes (hot path).  RICH: theta_v is a further variable (eq. 40).
// ------------------------------------------------------------------------------------------------
template <int Nq, bool MOIST, bool RICH> struct CmCfg11G {
  using C = CmCfg7<Nq, MOIST>;
  static constexpr int NF = C::NF, NP = C::NP, NV = C::NV, SLOT = C::SLOT, THREADS = C::THREADS;
  static constexpr int NS0 = C::NS;                     // u, v, w, h_tot, [q_t]
  static constexpr int NS = NS0 + (RICH ? 1 : 0);       // + theta_v (<= NV: the variables replace the state in place)
  static constexpr int NGEO = 15;                       // CmKP::geo fields 0..14
  static constexpr int NTR = NV + 1;                    // trace values per face node: state, z
  static constexpr int TS = C::fstride(NTR);
  static constexpr int OFF_Q = 0;                                        // [NV][SLOT]
  static constexpr int OFF_D = OFF_Q + NV * SLOT;                        // [3][NS][SLOT]
  static constexpr int OFF_GEO = OFF_D + 3 * NS * SLOT;                  // [NGEO][SLOT]
  static constexpr int OFF_T = OFF_GEO + NGEO * SLOT;                    // [6][TS]
  static constexpr int OFF_M = OFF_T + 5 * TS + NTR * NF + (NTR * NF & 1);
  static constexpr int DOUBLES = OFF_M + 2;
  static constexpr size_t SMEM = sizeof(double) * DOUBLES;
  static constexpr bool OK = SMEM <= 115712;
  static constexpr int MINB = C::cap(C::fit(SMEM), C::cap(896 / THREADS, 16));
  static_assert(NS <= NV, "gradient variables are stored in the state tiles");
};

template <int Nq, int NS, int SLOT, int D>
__device__ __forceinline__ void cm11_grad_line(const CmKP& p, const double* __restrict__ ss, double* __restrict__ dd, int l) {
  constexpr int NF = Nq * Nq, STR = Cm7Str<Nq, D>::value;
  const int b = l / Nq, a = l - b * Nq;
  const int base = (D == 0) ? Nq * l : (D == 1) ? a + NF * b : l;
#pragma unroll
  for (int v = 0; v < NS; ++v) {
    const double* in = ss + v * SLOT + base;
    double* out = dd + v * SLOT + base;
    double x[Nq];
#pragma unroll
    for (int m = 0; m < Nq; ++m) x[m] = in[m * STR];
#pragma unroll
    for (int i = 0; i < Nq; ++i) {
      double s = 0.0;
#pragma unroll
      for (int m = 0; m < Nq; ++m) s += p.D[i][m] * x[m];
      out[i * STR] = s;
    }
  }
}

template <int Nq, bool MOIST, bool RAW, bool RICH>
__global__ void __launch_bounds__(CmCfg7<Nq, MOIST>::THREADS, CmCfg11G<Nq, MOIST, RICH>::MINB) cm11_gradient_kernel(const __grid_constant__ CmKP p) {
  using C = CmCfg7<Nq, MOIST>;
  using R = CmCfg11G<Nq, MOIST, RICH>;
  constexpr int NF = C::NF, NP = C::NP, N = Nq - 1, NV = C::NV, SLOT = C::SLOT, NFP = C::NFP, THREADS = C::THREADS;
  constexpr int NS0 = R::NS0, NS = R::NS, TS = R::TS, NGEO = R::NGEO;
  extern __shared__ __align__(128) double smem11[];
  double* Qt = smem11 + R::OFF_Q;
  double* dt_ = smem11 + R::OFF_D;
  double* Gt = smem11 + R::OFF_GEO;
  double* T = smem11 + R::OFF_T;
  uint64_t* mbar = reinterpret_cast<uint64_t*>(smem11 + R::OFF_M);

  const int t = threadIdx.x;
  const Cm7Pos pos = cm7_position(p);
  const int e = pos.e;
  const int sh = C::ODD ? (e & 1) : 0;
  if (t == THREADS - 32) { cm7_mbar_init(mbar, 1); cm7_fence_mbar_init(); }
  __syncthreads();
  if (t == THREADS - 32) {
    const long long src = (long long)e * NP - sh;
    const uint32_t mb = cm7_saddr(mbar);
    cm7_mbar_expect_tx(mbar, (uint32_t)((NV + NGEO) * SLOT * sizeof(double)));
    uint32_t d = cm7_saddr(Qt);
#pragma unroll
    for (int v = 0; v < NV; ++v) { cm7_bulk_g2s_raw(d, p.Q + (size_t)v * p.stride + src, SLOT * 8, mb); d += SLOT * 8; }
    d = cm7_saddr(Gt);
#pragma unroll
    for (int k = 0; k < NGEO; ++k) { cm7_bulk_g2s_raw(d, p.geo + (size_t)k * p.stride + src, SLOT * 8, mb); d += SLOT * 8; }
  } else if (t > THREADS - 32 && p.ahead > 0 && e + p.ahead < p.Ne) {
    const int ea = e + p.ahead;
    const long long src = (long long)ea * NP - (C::ODD ? (ea & 1) : 0);
    for (int j = t - (THREADS - 32) - 1; j < NV + NGEO; j += 31)
      cm7_prefetch_l2((j < NV ? p.Q + (size_t)j * p.stride : p.geo + (size_t)(j - NV) * p.stride) + src, SLOT * 8);
  }
  for (int fn = THREADS - 1 - t; fn < 6 * NF; fn += THREADS) {   // neighbour traces: the thread that runs the face task copies them
    int f, m, d, s, nm, np_, kline;
    cm7_face_node<Nq>(fn, f, m, d, s, nm, np_, kline);
    if (!((pos.wallmask >> f) & 1)) {
      const size_t idp = (size_t)cm7_neighbour(p, pos, d, s) * NP + np_;
      double* dst = T + f * TS + m;
      const double* src = p.Q + idp;
#pragma unroll
      for (int v = 0; v < NV; ++v) { cm7_cp8(dst + v * NF, src); src += p.stride; }
      cm7_cp8(dst + NV * NF, p.geo + 10 * p.stride + idp);
    }
  }
  cm7_cp_commit();

  double* ss = Qt + sh; double* dd = dt_ + sh; const double* geo = Gt + sh;
  const int n = t;
  const bool node = t < NP;
  const int k_ = n / NF, j_ = (n - k_ * NF) / Nq, i_ = n - k_ * NF - j_ * Nq;
  cm7_mbar_wait(mbar, 0);

  // ---- phase 1: gradient variables of the own node, in place of the state
  if (node) {
    double Y[6], s[6];
#pragma unroll
    for (int v = 0; v < NV; ++v) Y[v] = ss[v * SLOT + n];
    cm7_eos_grad<MOIST, RICH>(p, Y, p.th.grav * geo[10 * SLOT + n], s);
#pragma unroll
    for (int v = 0; v < NS; ++v) ss[v * SLOT + n] = s[v];
  }
  cm7_cp_wait_all();
  __syncthreads();

  // ---- phase 2: face tasks (trace -> s* - s^-) and line tasks, independent
  for (int fn = THREADS - 1 - t; fn < 6 * NF; fn += THREADS) {
    int f, m, d, s, nm, np_, kline;
    cm7_face_node<Nq>(fn, f, m, d, s, nm, np_, kline);
    double* tr = T + f * TS + m;
    double dl[6];
    if (!((pos.wallmask >> f) & 1)) {
      double Yp[6], sp[6];
#pragma unroll
      for (int v = 0; v < NV; ++v) Yp[v] = tr[v * NF];
      cm7_eos_grad<MOIST, RICH>(p, Yp, p.th.grav * tr[NV * NF], sp);
#pragma unroll
      for (int v = 0; v < NS; ++v) dl[v] = 0.5 * (sp[v] - ss[v * SLOT + nm]);
    } else {
      // wall: u_bc = u^- - (n.u^-) n  (A6), n along Ja^d of the wall node; scalars unchanged (A8)
      const double A0 = geo[(3 * d) * SLOT + nm], A1 = geo[(3 * d + 1) * SLOT + nm], A2 = geo[(3 * d + 2) * SLOT + nm];
      const double ua = (ss[nm] * A0 + ss[SLOT + nm] * A1 + ss[2 * SLOT + nm] * A2) / (A0 * A0 + A1 * A1 + A2 * A2);
#pragma unroll
      for (int v = 0; v < NS; ++v) dl[v] = 0.0;
      dl[0] = -ua * A0; dl[1] = -ua * A1; dl[2] = -ua * A2;
    }
#pragma unroll
    for (int v = 0; v < NS; ++v) tr[v * NF] = dl[v];
  }
  for (int lt = t; lt < 3 * NFP; lt += THREADS) {
    const int d = lt / NFP, l = lt % NFP;
    if (l < NF) {
      if (d == 0) cm11_grad_line<Nq, NS, SLOT, 0>(p, ss, dd, l);
      else if (d == 1) cm11_grad_line<Nq, NS, SLOT, 1>(p, ss, dd + NS * SLOT, l);
      else cm11_grad_line<Nq, NS, SLOT, 2>(p, ss, dd + 2 * NS * SLOT, l);
    }
  }
  __syncthreads();

  // ---- phase 3: lifted jumps, physical gradient, closure, store
  if (node) {
    const size_t idx = (size_t)e * NP + n;
    double dr[6][3];
    const int c3[3] = {i_, j_, k_};
    const int m3[3] = {j_ + Nq * k_, i_ + Nq * k_, i_ + Nq * j_};
#pragma unroll
    for (int c = 0; c < 3; ++c) {
#pragma unroll
      for (int v = 0; v < NS; ++v) dr[v][c] = dd[(c * NS + v) * SLOT + n];
      if (c3[c] == 0 || c3[c] == N) {
        const bool hi = (c3[c] == N);
        const double* tr = T + (2 * c + (hi ? 1 : 0)) * TS + m3[c];
        const double w = hi ? p.inv_w0 : -p.inv_w0;
#pragma unroll
        for (int v = 0; v < NS; ++v) dr[v][c] += w * tr[v * NF];
      }
    }
    double Ja[3][3];
#pragma unroll
    for (int d = 0; d < 3; ++d)
#pragma unroll
      for (int c = 0; c < 3; ++c) Ja[d][c] = geo[(3 * d + c) * SLOT + n];
    const double invJ = geo[9 * SLOT + n];
    double G[6][3];
#pragma unroll
    for (int v = 0; v < NS; ++v)
#pragma unroll
      for (int c = 0; c < 3; ++c) G[v][c] = invJ * (Ja[0][c] * dr[v][0] + Ja[1][c] * dr[v][1] + Ja[2][c] * dr[v][2]);
    double Gr[5][3];
#pragma unroll
    for (int v = 0; v < 5; ++v)
#pragma unroll
      for (int c = 0; c < 3; ++c) Gr[v][c] = (v < NS0) ? G[v][c] : 0.0;
    double* o = p.Gout + idx;
    if (RAW) {
#pragma unroll
      for (int v = 0; v < 5; ++v)
#pragma unroll
        for (int c = 0; c < 3; ++c) __stcs(o + (size_t)(3 * v + c) * p.stride, Gr[v][c]);
    } else {
      double thv = 1.0, dthv = 0.0;
      if (RICH) { thv = ss[NS0 * SLOT + n]; dthv = G[NS0][2]; }
      double g[12];
      cm_closure<MOIST>(p, Gr, geo[11 * SLOT + n], geo[12 * SLOT + n], geo[13 * SLOT + n], geo[14 * SLOT + n], thv, dthv, g);
#pragma unroll
      for (int k = 0; k < C::NG; ++k) o[(size_t)k * p.stride] = g[k];
    }
  }
}
