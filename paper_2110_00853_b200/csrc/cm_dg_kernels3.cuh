// cm_dg_kernels3.cuh -- the hot kernels for flat bricks (GEOM == 0): persistent CTAs that sweep x-segments of
// elements through a TMA-fed shared-memory ring.
//
//   * Work unit = a segment of `seg_len` consecutive elements along x (consecutive in library order).  CTA b owns
//     units b, b + gridDim, ... and walks through them element by element; the grid is one wave of resident CTAs.
//   * The element's own fields (Q, and the packed SGS fluxes G in the tendency kernel) arrive by 1-D bulk TMA
//     (cp.async.bulk ... mbarrier::complete_tx) into a ring of S stage buffers, two elements ahead of the compute;
//     nobody waits on a global load of own data.  An element tile is NP*8 bytes; for odd NP it is fetched as
//     NP+1 doubles starting at the 16-byte boundary below it, so the data sit at offset (e & 1) of the slot.
//   * x-faces never touch global memory inside a segment: the +x neighbour is the next ring stage (already
//     landed), the -x neighbour's face plane was saved in shared memory by the previous iteration.  Only the y and
//     z neighbours' traces (runs of Nq and Nq^2 doubles) are gathered from L2, into registers, at the top of the
//     iteration, and only the 6 + 5 values per face node that the face-normal flux needs.  Everything those
//     gathers depend on (neighbour ids, z-table rows) is fetched one or two iterations ahead, so no warp ever
//     stalls on a dependent global load.
//   * Warp roles: NWN warps own the nodes (one thread per node: EOS, fluxes, assembly, update); every face is the
//     job of ONE warp with the face index a compile-time constant (warp 0: -x then +x, warps 1..: -y, +y, -z, +z),
//     one lane per face node; the tensor-product contractions are (line, variable) tasks over all warps with D as
//     constant-bank FMA operands.  The extra warp (no nodes) also prefetches the residual into L2.
//   * Phase order per element: fluxes -> lines (in place, saving the untouched face values) -> faces (which subtract
//     their lifted result from D_d F^d at the face node) -> assembly; four CTA barriers.
//   * The contravariant fluxes F^1, F^2 overwrite the G slots of the stage in place (same thread, same address),
//     F^3 and the face-value copies live in small work buffers: ~72 KB per CTA at N = 4, three CTAs per SM.
// Arithmetic follows cm_dg_physics.cuh (R12 pressure perturbation, MUFU-seeded rcp / sqrt).
#pragma once
#include <type_traits>
#include "cm_dg_internal.h"
#include "cm_dg_physics.cuh"

// ------------------------------------------------------------------------------------------------ PTX helpers
__device__ __forceinline__ uint32_t cm3_saddr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cm3_mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(cm3_saddr(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void cm3_mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(cm3_saddr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cm3_mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "LAB_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra LAB_WAIT;\n"
      "DONE:\n"
      "}\n" ::"r"(cm3_saddr(bar)), "r"(parity) : "memory");
}
// 1-D bulk TMA global -> shared, completion counted in bytes on an mbarrier (16-byte aligned src, dst, size)
__device__ __forceinline__ void cm3_bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(cm3_saddr(dst)),
               "l"(src), "r"(bytes), "r"(cm3_saddr(bar)) : "memory");
}
__device__ __forceinline__ void cm3_fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void cm3_fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void cm3_prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

template <int Nq, bool MOIST> struct CmCfg3 {
  static_assert(Nq * Nq <= 32, "one lane per face node");
  static constexpr int NF = Nq * Nq;
  static constexpr int NP = Nq * Nq * Nq;
  static constexpr int NV = MOIST ? 6 : 5;
  static constexpr int NG = MOIST ? 12 : 9;
  static constexpr int NS = MOIST ? 5 : 4;
  static constexpr int NGD = MOIST ? 5 : 4;                               // SGS values one face direction needs
  static constexpr int ODD = NP & 1;
  static constexpr int SLOT = NP + ODD;                                   // doubles per field tile in shared memory
  static constexpr int NWN = (NP + 31) / 32;                              // warps that own nodes
  static constexpr int NW = NWN + 1;
  static constexpr int THREADS = 32 * NW;
  static constexpr int GS = (NG > 2 * NV) ? NG : 2 * NV;                  // G region of a stage, reused for F^1, F^2
  static constexpr int ST_T = 3, ST_G = 4;                                // ring depth: tendency, gradient
  static constexpr int ZROW = (Nq + 2) * CM_ZTAB_W;                       // z-table rows: below, own Nq, above
  static constexpr int TEND_DOUBLES = ST_T * (NV + GS) * SLOT + NV * SLOT + SLOT + 6 * NV * NF + (2 * NV + 1) * NF + 2 * ZROW;
  static constexpr int GRAD_DOUBLES = ST_G * NV * SLOT + NS * SLOT + 3 * NS * SLOT + NS * 6 * NF + NS * NF + 2 * ZROW;
  static constexpr size_t TEND_SMEM = sizeof(double) * TEND_DOUBLES + 8 * ST_T;
  static constexpr size_t GRAD_SMEM = sizeof(double) * GRAD_DOUBLES + 8 * ST_G;
  static constexpr int fit(size_t smem) { return (int)((227 * 1024) / (smem + 1024)); }
  static constexpr int cap(int b, int hi) { return b < 1 ? 1 : (b > hi ? hi : b); }
  static constexpr int MINB_T = cap(fit(TEND_SMEM), 1536 / THREADS < 3 ? 1536 / THREADS : 3);
  static constexpr int MINB_G = cap(fit(GRAD_SMEM), 1536 / THREADS < 4 ? 1536 / THREADS : 4);
  // the warp that owns face f: 0 and 1 (x) on warp 0 (the -x task reads the plane the +x task then rewrites)
  __host__ __device__ static constexpr int face_warp(int f) { return f < 2 ? 0 : 1 + (f - 2) % (NW - 1); }
};

template <int F> using CmFace = std::integral_constant<int, F>;

__device__ __forceinline__ void cm3_site(const double* row, CmSite& s) {
  s.Phi = row[0]; s.rho_r = row[1]; s.rhoe_r = row[2]; s.rhoq_r = row[3]; s.E_r = row[4]; s.q_r = row[5]; s.icvm_r = row[6];
}

// primitives the gradient needs (u, v, w, h_tot, q): eq. (6)-(10), (13)-(14)
template <bool MOIST>
__device__ __forceinline__ void cm3_eos_grad(const CmKP& p, const double* Y, double Phi, double* s) {
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

// contravariant flux along axis D, A = s * e_D; gd = the SGS values that axis needs: tau(D,0..2), (J+D)_D, [d_q,D]
template <bool MOIST, bool SGS, int D>
__device__ __forceinline__ void cm3_flux_face(const double* Y, const CmPrim& P, const double* gd, double s, double* Fn) {
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

// index into the packed SGS array (tau xx,yy,zz,xy,xz,yz | J+D x,y,z | d_q x,y,z) of the k-th value axis d needs
__host__ __device__ constexpr int cm3_gidx(int d, int k) {
  return (k == 3) ? 6 + d : (k == 4) ? 9 + d : (k == d) ? d : k + d + 2;   // (0,1)->3, (0,2)->4, (1,2)->5
}

// own node / coincident neighbour node / their zeta indices of face F at face-node (a, b)
template <int Nq, int F>
__device__ __forceinline__ void cm3_face_nodes(int a, int b, int& nm, int& np_, int& km, int& kp) {
  constexpr int N = Nq - 1, NF = Nq * Nq, d = F >> 1, at = (F & 1) ? N : 0, ot = N - at;
  if (d == 0) { nm = at + Nq * a + NF * b; np_ = ot + Nq * a + NF * b; km = b; kp = b; }
  else if (d == 1) { nm = a + Nq * at + NF * b; np_ = a + Nq * ot + NF * b; km = b; kp = b; }
  else { nm = a + Nq * b + NF * at; np_ = a + Nq * b + NF * ot; km = at; kp = ot; }
}

struct Cm3Walk { int unit, off; };
__device__ __forceinline__ void cm3_advance(Cm3Walk& w, int L, int G) { if (++w.off == L) { w.off = 0; w.unit += G; } }
__device__ __forceinline__ int cm3_elem(const Cm3Walk& w, int L) { return w.unit * L + w.off; }

// z-table row a thread of the z-row loader needs for element e (row 0 = facing row of the -z neighbour, 1..Nq own,
// Nq+1 = facing row of the +z neighbour); -1 = none (wall)
template <int Nq>
__device__ __forceinline__ int cm3_zrow_of(const CmKP& p, int e, int t) {
  const int4 z = __ldg(reinterpret_cast<const int4*>(p.elz) + e);
  const int r = t / CM_ZTAB_W;
  return (r == 0) ? z.x : (r == Nq + 1) ? z.z : z.y + r - 1;
}

// ------------------------------------------------------------------------------------------------
// a3-a5: tendency + fused LSRK update (flat bricks)
// ------------------------------------------------------------------------------------------------
template <int Nq, bool MOIST, bool SGS>
__global__ void __launch_bounds__(CmCfg3<Nq, MOIST>::THREADS, CmCfg3<Nq, MOIST>::MINB_T) cm3_tendency_kernel(const __grid_constant__ CmKP p) {
  using C = CmCfg3<Nq, MOIST>;
  constexpr int NF = C::NF, NP = C::NP, N = Nq - 1, NV = C::NV, NG = C::NG, NGD = C::NGD, SLOT = C::SLOT, S = C::ST_T;
  constexpr int THREADS = C::THREADS, NW = C::NW;
  constexpr int STAGE = (NV + C::GS) * SLOT;
  extern __shared__ __align__(128) double smem3[];
  double* stage = smem3;                               // [S][NV + GS][SLOT]
  double* F3 = stage + S * STAGE;                      // [NV][SLOT]        F^3, then D_zeta F^3
  double* csh = F3 + NV * SLOT;                        // [SLOT]            sound speed
  double* ff = csh + SLOT;                             // [6][NV][NF]       untouched F^d on the six faces (saved by the line tasks)
  double* left = ff + 6 * NV * NF;                     // [2 NV + 1][NF]    Y, F^1, c on the +x plane of the previous element
  double* zrows = left + (2 * NV + 1) * NF;            // [2][ZROW]
  uint64_t* mbar = reinterpret_cast<uint64_t*>(zrows + 2 * C::ZROW);   // [S]

  const int t = threadIdx.x, warp = t >> 5, lane = t & 31;
  const int L = p.seg_len, G = gridDim.x;
  const int nitems = ((p.n_units - (int)blockIdx.x + G - 1) / G) * L;
  constexpr uint32_t tx_bytes = (uint32_t)((NV + (SGS ? NG : 0)) * SLOT * sizeof(double));

  auto issue = [&](const Cm3Walk& w, int s) {          // thread 0 only
    const long long e = (long long)w.unit * L + w.off;
    const long long src = e * NP - (C::ODD ? (e & 1) : 0);
    double* dst = stage + s * STAGE;
    cm3_mbar_expect_tx(&mbar[s], tx_bytes);
#pragma unroll
    for (int v = 0; v < NV; ++v) cm3_bulk_g2s(dst + v * SLOT, p.Q + v * p.stride + src, SLOT * 8, &mbar[s]);
    if (SGS)
#pragma unroll
      for (int k = 0; k < NG; ++k) cm3_bulk_g2s(dst + (NV + k) * SLOT, p.G + k * p.stride + src, SLOT * 8, &mbar[s]);
  };

  Cm3Walk wc{(int)blockIdx.x, 0}, wl{(int)blockIdx.x, 0};     // current item, item to load next
  if (t == 0) {
#pragma unroll
    for (int s = 0; s < S; ++s) cm3_mbar_init(&mbar[s], 1);
    cm3_fence_mbar_init();
  }
  __syncthreads();
  if (t == 0) {
    if (nitems > 0) { issue(wl, 0); cm3_advance(wl, L, G); }
    if (nitems > 1) { issue(wl, 1); cm3_advance(wl, L, G); }
  }

  // ---- per-thread constants
  const int n = t, nk = n / NF;
  const bool node = t < NP;
  const bool flane = lane < NF;
  const int la = lane % Nq, lb = (lane / Nq) % Nq;
  const int pf = (warp == 0) ? -1 : 1 + warp;          // primary (prefetched) face of this warp: 2..5, or none
  constexpr int NLT = 3 * NV * NF, LT_PER = (NLT + THREADS - 1) / THREADS;
  int loff[LT_PER], lstr[LT_PER], lff[LT_PER];
#pragma unroll
  for (int r = 0; r < LT_PER; ++r) {
    const int lt = t + r * THREADS;
    const int dv = lt / NF, l = lt % NF, d = dv / NV, v = dv % NV;
    const int base = (d == 0) ? Nq * l : (d == 1) ? (l % Nq) + NF * (l / Nq) : l;
    lstr[r] = (d == 0) ? 1 : (d == 1) ? Nq : NF;
    // offset relative to the stage base for d < 2 (slots NV + d*NV + v), or -(1 + offset in F3) for d == 2
    loff[r] = (lt >= NLT) ? 0x7fffffff : (d < 2) ? (NV + d * NV + v) * SLOT + base : -(1 + v * SLOT + base);
    lff[r] = ((2 * d) * NV + v) * NF + l;
  }

  // ---- software-pipelined lookups: neighbour ids one element ahead, z-table rows two / one ahead
  const bool zl = t < C::ZROW;
  Cm3Walk wn = wc; cm3_advance(wn, L, G);                     // item j+1
  int e = cm3_elem(wc, L);
  int nb_pf = -1, nb0 = -1, nb1 = -1;                         // neighbours of the current element
  int nb_pf_n = -1, nb0_n = -1, nb1_n = -1;                   // ... of the next element
  int zrow_n = -1;                                            // z-table row this thread loads for the next element
  if (nitems > 0) {
    if (pf >= 0 && pf < 6) nb_pf = __ldg(p.nbr + (size_t)e * 6 + pf);
    if (warp == 0) { nb0 = __ldg(p.nbr + (size_t)e * 6 + 0); nb1 = __ldg(p.nbr + (size_t)e * 6 + 1); }
    if (zl) {
      const int row = cm3_zrow_of<Nq>(p, e, t);
      zrows[t] = (row >= 0) ? __ldg(p.ztab + (size_t)row * CM_ZTAB_W + (t % CM_ZTAB_W)) : 0.0;
      if (nitems > 1) zrow_n = cm3_zrow_of<Nq>(p, cm3_elem(wn, L), t);
    }
  }
  __syncthreads();

  const bool stagemode = (p.mode != 0);
  const bool readres = stagemode && (p.rka != 0.0);

  int s_cur = 0; uint32_t ph_cur = 0;
  for (int j = 0; j < nitems; ++j) {
    const int sh = C::ODD ? (e & 1) : 0;
    double* own = stage + s_cur * STAGE + sh;
    const int s_nxt = (s_cur + 1 == S) ? 0 : s_cur + 1;
    const uint32_t ph_nxt = (s_cur + 1 == S) ? ph_cur ^ 1u : ph_cur;
    const bool has_next = (j + 1 < nitems);
    const int e_nxt = cm3_elem(wn, L);
    Cm3Walk wn2 = wn; cm3_advance(wn2, L, G);                 // item j+2
    const double* zr = zrows + (j & 1) * C::ZROW;

    // ---- top: TMA for item j+2 into the stage freed by iteration j-1; lookups for the next elements; gathers
    if (t == 0 && j + 2 < nitems) {
      const int s_ld = (s_nxt + 1 == S) ? 0 : s_nxt + 1;
      issue(wl, s_ld); cm3_advance(wl, L, G);
    }
    double zval = 0.0;
    if (has_next) {
      if (pf >= 0 && pf < 6) nb_pf_n = __ldg(p.nbr + (size_t)e_nxt * 6 + pf);
      if (warp == 0) { nb0_n = __ldg(p.nbr + (size_t)e_nxt * 6 + 0); nb1_n = __ldg(p.nbr + (size_t)e_nxt * 6 + 1); }
      if (zl) {
        if (zrow_n >= 0) zval = __ldg(p.ztab + (size_t)zrow_n * CM_ZTAB_W + (t % CM_ZTAB_W));
        zrow_n = (j + 2 < nitems) ? cm3_zrow_of<Nq>(p, cm3_elem(wn2, L), t) : -1;
      }
      if (warp == NW - 1 && readres) {                        // residual of the next element -> L2
        const double* base = p.dQ + (size_t)e_nxt * NP;
        constexpr int NL = (NP * 8 + 127) / 128 + 1;
        if (lane < NL)
#pragma unroll
          for (int v = 0; v < NV; ++v) cm3_prefetch_l2(base + v * p.stride + (16 * lane < NP ? 16 * lane : NP - 1));
      }
    }
    // neighbour trace of the primary face: 6 state values + the SGS values its normal flux needs
    double Yp[6], gp[5];
    auto gather = [&](auto Fc, int nb) {
      constexpr int F = decltype(Fc)::value, d = F >> 1;
      int nm, np_, km, kp; cm3_face_nodes<Nq, F>(la, lb, nm, np_, km, kp);
      const size_t idp = (size_t)nb * NP + np_;
#pragma unroll
      for (int v = 0; v < NV; ++v) Yp[v] = __ldg(p.Q + v * p.stride + idp);
      if (SGS)
#pragma unroll
        for (int k = 0; k < NGD; ++k) gp[k] = __ldg(p.G + (size_t)cm3_gidx(d, k) * p.stride + idp);
    };
    if (flane && nb_pf >= 0) {
      if (pf == 2) gather(CmFace<2>{}, nb_pf);
      else if (pf == 3) gather(CmFace<3>{}, nb_pf);
      else if (pf == 4) gather(CmFace<4>{}, nb_pf);
      else if (pf == 5) gather(CmFace<5>{}, nb_pf);
    }

    cm3_mbar_wait(&mbar[s_cur], ph_cur);

    // ---- phase 0: primitives and contravariant fluxes of the own node
    double buoy = 0.0;
    if (node) {
      double Y[6], g[12]; CmSite st; CmPrim P;
#pragma unroll
      for (int v = 0; v < NV; ++v) Y[v] = own[v * SLOT + n];
      if (SGS)
#pragma unroll
        for (int k = 0; k < NG; ++k) g[k] = own[(NV + k) * SLOT + n];
      cm3_site(zr + (1 + nk) * CM_ZTAB_W, st);
      cm_eos<MOIST>(p, Y, st, P);
      buoy = P.drho * p.th.grav;
      csh[n] = cm_sqrt(P.c2);
      double Fa[6];
      cm_flux_axis<MOIST, 0>(Y, P, SGS, g, p.cA[0], Fa);
#pragma unroll
      for (int v = 0; v < NV; ++v) own[(NV + v) * SLOT + n] = Fa[v];
      cm_flux_axis<MOIST, 1>(Y, P, SGS, g, p.cA[1], Fa);
#pragma unroll
      for (int v = 0; v < NV; ++v) own[(2 * NV + v) * SLOT + n] = Fa[v];
      cm_flux_axis<MOIST, 2>(Y, P, SGS, g, p.cA[2], Fa);
#pragma unroll
      for (int v = 0; v < NV; ++v) F3[v * SLOT + n] = Fa[v];
    }
    __syncthreads();

    // ---- phase 1: (line, variable) tasks, F^d <- D_d F^d in place, end values saved for the face tasks;
    //      the residual is fetched meanwhile
    const size_t idx = (size_t)e * NP + n;
    double dold[6];
    if (node)
#pragma unroll
      for (int v = 0; v < NV; ++v) dold[v] = readres ? __ldcs(p.dQ + v * p.stride + idx) : 0.0;   // streaming: keep L2 for Q / G traces
#pragma unroll
    for (int r = 0; r < LT_PER; ++r) {
      if (loff[r] != 0x7fffffff) {
        double* a = (loff[r] >= 0) ? own + loff[r] : F3 + (-loff[r] - 1);
        const int str = lstr[r];
        double x[Nq], y[Nq];
#pragma unroll
        for (int m = 0; m < Nq; ++m) x[m] = a[m * str];
        ff[lff[r]] = x[0]; ff[lff[r] + NV * NF] = x[N];
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
    __syncthreads();

    // ---- phase 2: face tasks.  r = sgn F^- . A - sJ F*;  D_d F^d at the face node -= r / w_0
    auto face = [&](auto Fc, int nb, int src) {          // src: 0 gathered registers, 1 next ring stage, 2 `left`, 3 load now
      constexpr int F = decltype(Fc)::value, d = F >> 1;
      constexpr double sgn = (F & 1) ? 1.0 : -1.0;
      int nm, np_, km, kp; cm3_face_nodes<Nq, F>(la, lb, nm, np_, km, kp);
      const double sJ = p.cA[d], A = sgn * sJ;
      double Ym[6], Ftm[6], r[6];
#pragma unroll
      for (int v = 0; v < NV; ++v) { Ym[v] = own[v * SLOT + nm]; Ftm[v] = sgn * ff[(F * NV + v) * NF + lane]; }
      const double cm_ = csh[nm];
      const double uAm = (Ym[1 + d] * A) * cm_rcp(Ym[0]);                    // sJ (u^- . n)
      if (F == 1) {                                      // save the +x plane for the next element's -x face
#pragma unroll
        for (int v = 0; v < NV; ++v) { left[v * NF + lane] = Ym[v]; left[(NV + v) * NF + lane] = Ftm[v]; }
        left[2 * NV * NF + lane] = cm_;
      }
      if (nb >= 0) {
        double Fp[6], cp, uAp;
        if (src == 2) {
#pragma unroll
          for (int v = 0; v < NV; ++v) { Yp[v] = left[v * NF + lane]; Fp[v] = sgn * left[(NV + v) * NF + lane]; }
          cp = left[2 * NV * NF + lane];
          uAp = (Yp[1 + d] * A) * cm_rcp(Yp[0]);
        } else {
          if (src == 1) {
            cm3_mbar_wait(&mbar[s_nxt], ph_nxt);
            const double* nx = stage + s_nxt * STAGE + (C::ODD ? (e_nxt & 1) : 0) + np_;
#pragma unroll
            for (int v = 0; v < NV; ++v) Yp[v] = nx[v * SLOT];
            if (SGS)
#pragma unroll
              for (int k = 0; k < NGD; ++k) gp[k] = nx[(NV + cm3_gidx(d, k)) * SLOT];
          } else if (src == 3) {
            const size_t idp = (size_t)nb * NP + np_;
#pragma unroll
            for (int v = 0; v < NV; ++v) Yp[v] = __ldg(p.Q + v * p.stride + idp);
            if (SGS)
#pragma unroll
              for (int k = 0; k < NGD; ++k) gp[k] = __ldg(p.G + (size_t)cm3_gidx(d, k) * p.stride + idp);
          }
          CmSite st; CmPrim P;
          constexpr int zrow_c = (F == 4) ? 0 : Nq + 1;
          cm3_site(zr + ((F < 4) ? 1 + km : zrow_c) * CM_ZTAB_W, st);
          cm_eos<MOIST>(p, Yp, st, P);
          cm3_flux_face<MOIST, SGS, d>(Yp, P, gp, A, Fp);
          cp = cm_sqrt(P.c2);
          uAp = A * ((d == 0) ? P.u : (d == 1) ? P.v : P.w);
        }
        const double lamsJ = fmax(fabs(uAm) + cm_ * sJ, fabs(uAp) + cp * sJ);      // sJ * lambda (R2)
#pragma unroll
        for (int v = 0; v < NV; ++v) r[v] = 0.5 * (Ftm[v] - Fp[v]) - 0.5 * lamsJ * (Ym[v] - Yp[v]);
      } else {
        // free-slip wall (A6-A7): Rusanov against the mirrored state = [0; (p' + rho u_n (u_n + lambda)) n; 0; 0];
        // second-order normal fluxes vanish (R10) except the prescribed bottom energy flux
        CmSite st; CmPrim P;
        cm3_site(zr + (1 + km) * CM_ZTAB_W, st);
        cm_eos<MOIST>(p, Ym, st, P);
        const double un = uAm / sJ;
        const double lam = fabs(un) + cm_;
        const double mom = P.pp + Ym[0] * un * (un + lam);
#pragma unroll
        for (int v = 0; v < NV; ++v) r[v] = Ftm[v];
        r[1 + d] -= mom * A;
        if (F == 4) r[4] += sJ * p.shf;
      }
      double* Fd = ((d == 2) ? F3 : own + (NV + d * NV) * SLOT) + nm;
#pragma unroll
      for (int v = 0; v < NV; ++v) Fd[v * SLOT] -= p.inv_w0 * r[v];
    };
    if (warp == 0) {
      if (flane) {
        face(CmFace<0>{}, nb0, (wc.off > 0 && nb0 == e - 1) ? 2 : 3);       // -x first: it reads `left`, +x rewrites it
        face(CmFace<1>{}, nb1, (has_next && wc.off + 1 < L && nb1 == e + 1) ? 1 : 3);
      }
    } else {
#pragma unroll
      for (int f = 2; f < 6; ++f) {
        if (C::face_warp(f) == warp && flane) {
          const int nb = (f == pf) ? nb_pf : __ldg(p.nbr + (size_t)e * 6 + f);
          const int src = (f == pf) ? 0 : 3;
          if (f == 2) face(CmFace<2>{}, nb, src);
          else if (f == 3) face(CmFace<3>{}, nb, src);
          else if (f == 4) face(CmFace<4>{}, nb, src);
          else face(CmFace<5>{}, nb, src);
        }
      }
    }
    __syncthreads();

    // ---- phase 3: assemble the tendency of the own node and update
    if (node) {
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        const double a = own[(NV + v) * SLOT + n] + own[(2 * NV + v) * SLOT + n] + F3[v * SLOT + n];
        double rhs = -p.invJ * a;
        if (v == 3) rhs -= buoy;                                   // -(rho - rho_r) grad Phi   (eq. 4)
        if (!stagemode) {
          __stcs(p.dQ + v * p.stride + idx, rhs);
        } else {
          // a5: dU <- A_s dU + dt RHS ; U <- U + B_s dU
          const double dnew = p.rka * dold[v] + p.dt * rhs;
          __stcs(p.dQ + v * p.stride + idx, dnew);
          __stcs(p.Qnew + v * p.stride + idx, own[v * SLOT + n] + p.rkb * dnew);
        }
      }
    }
    if (zl && has_next) zrows[((j + 1) & 1) * C::ZROW + t] = zval;
    cm3_fence_proxy_async();      // generic-proxy accesses of this stage are ordered before the TMA refill
    __syncthreads();

    wc = wn; wn = wn2; e = e_nxt; s_cur = s_nxt; ph_cur = ph_nxt;
    nb_pf = nb_pf_n; nb0 = nb0_n; nb1 = nb1_n;
  }
}

// ------------------------------------------------------------------------------------------------
// a2: auxiliary gradient + Smagorinsky-Lilly (flat bricks)
// ------------------------------------------------------------------------------------------------
template <int Nq, bool MOIST>
__global__ void __launch_bounds__(CmCfg3<Nq, MOIST>::THREADS, CmCfg3<Nq, MOIST>::MINB_G) cm3_gradient_kernel(const __grid_constant__ CmKP p) {
  using C = CmCfg3<Nq, MOIST>;
  constexpr int NF = C::NF, NP = C::NP, N = Nq - 1, NV = C::NV, NS = C::NS, SLOT = C::SLOT, S = C::ST_G, THREADS = C::THREADS;
  constexpr int STAGE = NV * SLOT;
  extern __shared__ __align__(128) double smem3[];
  double* stage = smem3;                               // [S][NV][SLOT]
  double* s_sh = stage + S * STAGE;                    // [NS][SLOT]       gradient variables u, v, w, h_tot, [q]
  double* d_sh = s_sh + NS * SLOT;                     // [3][NS][SLOT]    reference-space derivatives
  double* fbuf = d_sh + 3 * NS * SLOT;                 // [NS][6*NF]       s* - s^- per face node
  double* left = fbuf + NS * 6 * NF;                   // [NS][NF]         s on the +x plane of the previous element
  double* zrows = left + NS * NF;                      // [2][ZROW]
  uint64_t* mbar = reinterpret_cast<uint64_t*>(zrows + 2 * C::ZROW);

  const int t = threadIdx.x, warp = t >> 5, lane = t & 31;
  const int L = p.seg_len, G = gridDim.x;
  const int nitems = ((p.n_units - (int)blockIdx.x + G - 1) / G) * L;

  auto issue = [&](const Cm3Walk& w, int s) {
    const long long e = (long long)w.unit * L + w.off;
    const long long src = e * NP - (C::ODD ? (e & 1) : 0);
    double* dst = stage + s * STAGE;
    cm3_mbar_expect_tx(&mbar[s], (uint32_t)(NV * SLOT * sizeof(double)));
#pragma unroll
    for (int v = 0; v < NV; ++v) cm3_bulk_g2s(dst + v * SLOT, p.Q + v * p.stride + src, SLOT * 8, &mbar[s]);
  };

  Cm3Walk wc{(int)blockIdx.x, 0}, wl{(int)blockIdx.x, 0};
  if (t == 0) {
#pragma unroll
    for (int s = 0; s < S; ++s) cm3_mbar_init(&mbar[s], 1);
    cm3_fence_mbar_init();
  }
  __syncthreads();
  if (t == 0)
    for (int s = 0; s < S - 1; ++s)
      if (s < nitems) { issue(wl, s); cm3_advance(wl, L, G); }

  const int n = t, ni = n % Nq, nj = (n / Nq) % Nq, nk = n / NF;
  const bool node = t < NP;
  const bool flane = lane < NF;
  const int la = lane % Nq, lb = (lane / Nq) % Nq;
  const int pf = (warp == 0) ? -1 : 1 + warp;
  constexpr int NLT = 3 * NS * NF, LT_PER = (NLT + THREADS - 1) / THREADS;
  int lin[LT_PER], lstr[LT_PER];
#pragma unroll
  for (int r = 0; r < LT_PER; ++r) {
    const int lt = t + r * THREADS;
    const int dv = lt / NF, l = lt % NF, d = dv / NS, v = dv % NS;
    const int base = (d == 0) ? Nq * l : (d == 1) ? (l % Nq) + NF * (l / Nq) : l;
    lstr[r] = (d == 0) ? 1 : (d == 1) ? Nq : NF;
    lin[r] = (lt >= NLT) ? -1 : ((d * NS + v) << 16) | (v * SLOT + base);     // output slot d*NS+v | input offset in s_sh
  }

  const bool zl = t < C::ZROW;
  Cm3Walk wn = wc; cm3_advance(wn, L, G);
  int e = cm3_elem(wc, L);
  int nb_pf = -1, nb0 = -1, nb1 = -1, nb_pf_n = -1, nb0_n = -1, nb1_n = -1, zrow_n = -1;
  if (nitems > 0) {
    if (pf >= 0 && pf < 6) nb_pf = __ldg(p.nbr + (size_t)e * 6 + pf);
    if (warp == 0) { nb0 = __ldg(p.nbr + (size_t)e * 6 + 0); nb1 = __ldg(p.nbr + (size_t)e * 6 + 1); }
    if (zl) {
      const int row = cm3_zrow_of<Nq>(p, e, t);
      zrows[t] = (row >= 0) ? __ldg(p.ztab + (size_t)row * CM_ZTAB_W + (t % CM_ZTAB_W)) : 0.0;
      if (nitems > 1) zrow_n = cm3_zrow_of<Nq>(p, cm3_elem(wn, L), t);
    }
  }
  __syncthreads();

  int s_cur = 0; uint32_t ph_cur = 0;
  for (int j = 0; j < nitems; ++j) {
    const int sh = C::ODD ? (e & 1) : 0;
    const double* own = stage + s_cur * STAGE + sh;
    const int s_nxt = (s_cur + 1 == S) ? 0 : s_cur + 1;
    const uint32_t ph_nxt = (s_cur + 1 == S) ? ph_cur ^ 1u : ph_cur;
    const bool has_next = (j + 1 < nitems);
    const int e_nxt = cm3_elem(wn, L);
    Cm3Walk wn2 = wn; cm3_advance(wn2, L, G);
    const double* zr = zrows + (j & 1) * C::ZROW;

    if (t == 0 && j + S - 1 < nitems) {
      const int s_ld = (s_cur == 0) ? S - 1 : s_cur - 1;          // the stage iteration j-1 used
      issue(wl, s_ld); cm3_advance(wl, L, G);
    }
    double zval = 0.0;
    if (has_next) {
      if (pf >= 0 && pf < 6) nb_pf_n = __ldg(p.nbr + (size_t)e_nxt * 6 + pf);
      if (warp == 0) { nb0_n = __ldg(p.nbr + (size_t)e_nxt * 6 + 0); nb1_n = __ldg(p.nbr + (size_t)e_nxt * 6 + 1); }
      if (zl) {
        if (zrow_n >= 0) zval = __ldg(p.ztab + (size_t)zrow_n * CM_ZTAB_W + (t % CM_ZTAB_W));
        zrow_n = (j + 2 < nitems) ? cm3_zrow_of<Nq>(p, cm3_elem(wn2, L), t) : -1;
      }
    }
    double Yp[6];
    auto gather = [&](auto Fc, int nb) {
      constexpr int F = decltype(Fc)::value;
      int nm, np_, km, kp; cm3_face_nodes<Nq, F>(la, lb, nm, np_, km, kp);
      const size_t idp = (size_t)nb * NP + np_;
#pragma unroll
      for (int v = 0; v < NV; ++v) Yp[v] = __ldg(p.Q + v * p.stride + idp);
    };
    if (flane && nb_pf >= 0) {
      if (pf == 2) gather(CmFace<2>{}, nb_pf);
      else if (pf == 3) gather(CmFace<3>{}, nb_pf);
      else if (pf == 4) gather(CmFace<4>{}, nb_pf);
      else if (pf == 5) gather(CmFace<5>{}, nb_pf);
    }

    cm3_mbar_wait(&mbar[s_cur], ph_cur);

    // ---- phase 0: gradient variables of the own node
    if (node) {
      double Y[6], s[5];
#pragma unroll
      for (int v = 0; v < NV; ++v) Y[v] = own[v * SLOT + n];
      cm3_eos_grad<MOIST>(p, Y, zr[(1 + nk) * CM_ZTAB_W], s);
#pragma unroll
      for (int v = 0; v < NS; ++v) s_sh[v * SLOT + n] = s[v];
    }
    __syncthreads();

    // ---- phase 1: face tasks (s* - s^-) and line tasks (reference-space derivatives); both only read s_sh
    auto face = [&](auto Fc, int nb, int src) {          // src: 0 gathered registers, 1 next ring stage, 2 `left`, 3 load now
      constexpr int F = decltype(Fc)::value, d = F >> 1;
      constexpr double sgn = (F & 1) ? 1.0 : -1.0;
      int nm, np_, km, kp; cm3_face_nodes<Nq, F>(la, lb, nm, np_, km, kp);
      double sm[5], dl[5];
#pragma unroll
      for (int v = 0; v < NS; ++v) sm[v] = s_sh[v * SLOT + nm];
      if (F == 1)
#pragma unroll
        for (int v = 0; v < NS; ++v) left[v * NF + lane] = sm[v];
      if (nb >= 0) {
        if (src == 2) {
#pragma unroll
          for (int v = 0; v < NS; ++v) dl[v] = 0.5 * (left[v * NF + lane] - sm[v]);
        } else {
          if (src == 1) {
            cm3_mbar_wait(&mbar[s_nxt], ph_nxt);
            const double* nx = stage + s_nxt * STAGE + (C::ODD ? (e_nxt & 1) : 0) + np_;
#pragma unroll
            for (int v = 0; v < NV; ++v) Yp[v] = nx[v * SLOT];
          } else if (src == 3) {
            const size_t idp = (size_t)nb * NP + np_;
#pragma unroll
            for (int v = 0; v < NV; ++v) Yp[v] = __ldg(p.Q + v * p.stride + idp);
          }
          constexpr int zrow_c = (F == 4) ? 0 : Nq + 1;
          double sp[5];
          cm3_eos_grad<MOIST>(p, Yp, zr[((F < 4) ? 1 + km : zrow_c) * CM_ZTAB_W], sp);
#pragma unroll
          for (int v = 0; v < NS; ++v) dl[v] = 0.5 * (sp[v] - sm[v]);
        }
      } else {
        // wall: u_bc = u^- - (n.u^-) n  (A6); scalars unchanged (A8)
        const double A = sgn * p.cA[d];
        const double ua = (sm[d] * A) / (A * A);
#pragma unroll
        for (int v = 0; v < NS; ++v) dl[v] = (v == d) ? -ua * A : 0.0;
      }
#pragma unroll
      for (int v = 0; v < NS; ++v) fbuf[v * 6 * NF + F * NF + lane] = dl[v];
    };
    if (warp == 0) {
      if (flane) {
        face(CmFace<0>{}, nb0, (wc.off > 0 && nb0 == e - 1) ? 2 : 3);
        face(CmFace<1>{}, nb1, (has_next && wc.off + 1 < L && nb1 == e + 1) ? 1 : 3);
      }
    } else {
#pragma unroll
      for (int f = 2; f < 6; ++f) {
        if (C::face_warp(f) == warp && flane) {
          const int nb = (f == pf) ? nb_pf : __ldg(p.nbr + (size_t)e * 6 + f);
          const int src = (f == pf) ? 0 : 3;
          if (f == 2) face(CmFace<2>{}, nb, src);
          else if (f == 3) face(CmFace<3>{}, nb, src);
          else if (f == 4) face(CmFace<4>{}, nb, src);
          else face(CmFace<5>{}, nb, src);
        }
      }
    }
#pragma unroll
    for (int r = 0; r < LT_PER; ++r) {
      if (lin[r] >= 0) {
        const double* in = s_sh + (lin[r] & 0xffff);
        double* out = d_sh + (lin[r] >> 16) * SLOT + ((lin[r] & 0xffff) % SLOT);
        const int str = lstr[r];
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
    __syncthreads();

    // ---- phase 2: physical gradient of the own node, closure, store
    if (node) {
      const size_t idx = (size_t)e * NP + n;
      const double w0i = p.inv_w0;
      double Gr[5][3];
#pragma unroll
      for (int v = 0; v < NS; ++v) {
        double dr = d_sh[(0 * NS + v) * SLOT + n], ds = d_sh[(1 * NS + v) * SLOT + n], dt = d_sh[(2 * NS + v) * SLOT + n];
        const double* fb = fbuf + v * 6 * NF;
        if (ni == 0) dr -= w0i * fb[0 * NF + nj + Nq * nk];
        if (ni == N) dr += w0i * fb[1 * NF + nj + Nq * nk];
        if (nj == 0) ds -= w0i * fb[2 * NF + ni + Nq * nk];
        if (nj == N) ds += w0i * fb[3 * NF + ni + Nq * nk];
        if (nk == 0) dt -= w0i * fb[4 * NF + ni + Nq * nj];
        if (nk == N) dt += w0i * fb[5 * NF + ni + Nq * nj];
        Gr[v][0] = (p.cA[0] * p.invJ) * dr; Gr[v][1] = (p.cA[1] * p.invJ) * ds; Gr[v][2] = (p.cA[2] * p.invJ) * dt;
      }
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
        __stcs(o, m2nu * Sxx); __stcs(o + st, m2nu * Syy); __stcs(o + 2 * st, m2nu * Szz);
        __stcs(o + 3 * st, m2nu * Sxy); __stcs(o + 4 * st, m2nu * Sxz); __stcs(o + 5 * st, m2nu * Syz);
        __stcs(o + 6 * st, mDt * Gr[3][0]); __stcs(o + 7 * st, mDt * Gr[3][1]); __stcs(o + 8 * st, mDt * Gr[3][2]);
        if (MOIST) { __stcs(o + 9 * st, mDt * Gr[4][0]); __stcs(o + 10 * st, mDt * Gr[4][1]); __stcs(o + 11 * st, mDt * Gr[4][2]); }
      }
    }
    if (zl && has_next) zrows[((j + 1) & 1) * C::ZROW + t] = zval;
    __syncthreads();

    wc = wn; wn = wn2; e = e_nxt; s_cur = s_nxt; ph_cur = ph_nxt;
    nb_pf = nb_pf_n; nb0 = nb0_n; nb1 = nb1_n;
  }
}
