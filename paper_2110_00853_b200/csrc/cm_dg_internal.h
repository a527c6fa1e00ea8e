// cm_dg_internal.h -- shared declarations of the CUDA implementation behind include/cm_dg.h.
// Not part of the public boundary.  P:L<n> = line of the paper text.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#define CM_MAXNQ 8
#define CM_ZTAB_W 8   // doubles per z-table row (flat meshes): Phi, rho_r, rhoe_r, rhoq_r, E_r, q_r, 1/c_vm_r, tau_s (sponge)
#define CM_NGEO 16    // general geometry, per node: Ja[9], 1/J, z, (C_s Delta)^2, Delta_m^2 [3], tau_s (sponge)

// Thermodynamic constants of eq. (7)-(14) in the combinations the kernels use.
struct CmThermo {
  double R_d, c_vd;
  double a;    // R_v - R_d
  double b;    // c_vv - c_vd
  double T_0, I_v0, grav;
  double dk;   // a c_vd - R_d b   (numerator of kappa - kappa_r, reading R12)
  double icvd, kappa_d;  // 1 / c_vd, R_d / c_vd (dry air)
  double p_0, kap_pd, iRd;   // theta_v = (p / (rho R_d)) (p_0 / p)^(R_d / c_pd)   (eq. 40, reading R25)
  // saturation adjustment (eq. 15; stored-metric kernels): p*(T) = p_tr (T / T_tr)^sx1 exp(sx2 (1 / T_tr - 1 / T))
  double R_v, c_vv, c_vl, Lv0, dcp;   // L(T) = Lv0 + dcp (T - T_0), dcp = c_vv + R_v - c_vl
  double p_tr, iT_tr, sx1, sx2;       // sx1 = dcp / R_v, sx2 = (Lv0 - dcp T_0) / R_v
};

// Kernel argument block (passed by value, lives in the constant bank).
struct CmKP {
  // sizes
  int Ne;                // elements
  // tiled element order e = ((((ey / gPY) * gNXC + ex / gL) * gEz + ez) * gPY + ey % gPY) * gL + ex % gL
  int gL, gPY, gNXC, gNYP, gEz;   // x-chunk length (divides Ex), y-patch height (divides Ey), Ex / gL, Ey / gPY, Ez
  int gbc[3];            // per direction: 1 = walls, 0 = periodic
  int gS;                // row-sweep kernels: elements per row (divides gL)
  int ahead;             // flat: L2 prefetch distance in elements of the launch order (0 = off)
  float ginvL, ginvNXC;  // 1 / gL, 1 / gNXC (exact small-integer division in cm7_position)
  long long stride;      // field stride in doubles
  int sgs;               // 0 inviscid | 1 Smagorinsky-Lilly | 2 Vreman
  int richardson;        // eq. (40): nu_t *= f_b (one more gradient variable, theta_v)
  int riemann;           // 0 Rusanov | 1 HLLC | 2 Roe (stored-metric kernels)
  int use_ref;           // reference state removed (R12) or plain pressure
  int terrain;           // stored-metric meshes: 1 = terrain-following (geom == 1): Ja^1, Ja^2 axis-aligned (cm_dg_kernels11.cuh)
  int satadj;            // 1: temperature and liquid water from the saturation adjustment of eq. (15) (stored-metric kernels)
  int mode;              // tendency: 0 dQ := rhs | 1 LSRK stage.  gradient: 0 packed SGS fluxes | 1 raw 15 gradients
  // arrays
  const double* Q;       // [nvar][stride]
  const double* G;       // packed SGS fluxes [ngrad][stride] (tendency input)
  double* Gout;          // gradient output
  double* dQ;            // residual (in/out) or rhs output
  double* Qnew;          // LSRK: updated state (ping-pong buffer)
  const int* nbr;        // [Ne][6] neighbour in library order, <0 = wall (stored-metric kernels; the flat ones compute it)
  const int* erow;       // flat: [Ne] first z-table row of the element (= ez*Nq)
  const double* ztab;    // flat: [Ez*Nq][CM_ZTAB_W]
  const double* geo;     // general: [CM_NGEO][stride]
  const double* ref;     // general: [3][stride] rho_r, rhoe_r, rhoq_r
  // constants
  CmThermo th;
  double cA[3];          // flat: Ja^d_d = h_e h_f / 4
  double invJ;           // flat: 8 / (hx hy hz)
  double cs2delta2;      // flat: (C_s Delta)^2
  double cs2;            // C_s^2
  double d2[3];          // flat: squared mixing lengths Delta_m^2 = (h_m / N)^2 of the Vreman model (eq. 39c)
  double urelax[3];      // Rayleigh sponge: relaxation velocity (eq. A4); tau_s comes with the z table / geometry
  double inv_Pr;
  double shf;            // prescribed upward energy flux at the bottom wall: SHF + LHF
  double evap;           // prescribed evaporation E through the bottom wall [kg m^-2 s^-1]
  double drag_cd;        // drag coefficient C_d of eq. (A2) on the bottom wall, 0 = free slip
  double inv_w0;         // 1 / w_0 = N (N+1) / 2
  double rka, rkb, dt;   // LSRK stage coefficients
  double D[CM_MAXNQ][CM_MAXNQ];  // D[i][m] = L_m'(xi_i)
};

struct CmLaunchCfg { int epb; int threads; size_t smem_grad; size_t smem_tend; };

// implemented in cm_dg_kernels_inst.cu (one object per polynomial order)
// variant: 2 = thread-per-node kernels (cm_dg_kernels2.cuh; any geometry), 7 = CTA-per-element kernels fed by bulk TMA
// and cp.async (cm_dg_kernels7.cuh; flat bricks)
typedef cudaError_t (*cm_launch_fn)(const CmKP& kp, int moist, int general, int variant, cudaStream_t st);
#define CM_DECL_LAUNCHERS(NQ)                                                                 \
  cudaError_t cm_launch_gradient_nq##NQ(const CmKP& kp, int moist, int general, int variant, cudaStream_t st); \
  cudaError_t cm_launch_tendency_nq##NQ(const CmKP& kp, int moist, int general, int variant, cudaStream_t st);
CM_DECL_LAUNCHERS(3)
CM_DECL_LAUNCHERS(4)
CM_DECL_LAUNCHERS(5)
CM_DECL_LAUNCHERS(6)
CM_DECL_LAUNCHERS(7)
CM_DECL_LAUNCHERS(8)
