// dg_oracle.cpp -- CPU ORACLE for the nodal-DG right-hand side of arXiv 2110.00853 (ClimateMachine LES).
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
// cpu_baseline / --impl reference legs of bench.py may load it.  It shares no code, header, table or
// constant generator with the CUDA path under paper_2110_00853_b200/csrc/.
//
// Plain, slow, fp64, written step by step from the paper (P:L<n> = /root/reference/PAPER.md line):
//   O1  LGL nodes / weights / derivative matrix            P:L202-204, eq. (21)-(23) P:L223-228
//   O2  brick mesh, linear-decay terrain warp, metric terms P:L186-190, eq. (24)
//   O3  thermodynamics (dry / non-condensing moist air)    eq. (6), (7)-(10) P:L100-134, (13)-(14) P:L154-160
//   O4  BR1 auxiliary gradient with central flux           eq. (28)-(31) P:L262-274, (A6)-(A8) P:L708-714
//   O5  Smagorinsky-Lilly closure                          eq. (33)-(38) P:L296-326
//   O6  fluxes F1, F2 and source S                         eq. (1),(2),(4),(5),(16) P:L54-95
//   O7  weak-form tendency (eq. 26) and the strong form (eq. 32)
//   O8  Rusanov flux (eq. 27), central flux for F2, walls (App. A)
//   O9  LSRK54 (Carpenter & Kennedy 1994, cited P:L286) and forward Euler
//   O10 diagnostics: eq. (57), (61)-(62) P:L587-591
//   O11 Vreman eddy viscosity (eq. 39a-d) and the Richardson stability factor (eq. 40)
//   O12 Rayleigh sponge (eq. A4-A5) and the exponential element filter (eq. 52)
//   O13 any 2N-storage LSRK coefficient table, HLLC and Roe fluxes (named P:L256; textbook forms),
//       curl-invariant metric terms (Kopriva 2006) for fully 3-D warps
//   O15 saturation adjustment (eq. 15): Newton iteration for T with the closed-form saturation vapour pressure
//       of a calorically perfect gas (Romps 2008, cited P:L172); warm phase (liquid condensate) -- reading R31
//   O14 surface fluxes at the bottom wall: aerodynamic drag law (eq. A2), prescribed evaporation and latent
//       heat flux; density-weighted horizontal statistics (eq. B1-B4)
// Readings of the paper where it is silent or garbled are R1..R29 of DESIGN.md.
//
// Data layout of the oracle (deliberately NOT the GPU layout): array-of-structures,
//   Q[e][n][v], e = ex + Ex*(ey + Ey*ez) lexicographic, n = i + Nq*(j + Nq*k), v = rho,rhou,rhov,rhow,rhoe,[rhoq].
// Parity status: every function here is pinned by tests/test_oracle_*.py except the conventions
// R2, R6, R7, R8, R11 (lambda, per-side nu_t, filter width, slab y-extent, constants), which the paper
// does not fix: "parity unpinned" for those choices only.
//
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC dg_oracle.cpp -o liboracle_dg.so

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr int MAXNQ = 9;

struct Ctx {
  int N, Nq, Np;
  int ne[3];
  int64_t Ne;
  double lo[3], hi[3];
  int bc[3];
  int nvar;
  int geom;
  std::vector<double> zsfc;   // geom==1: [Ey*Nq][Ex*Nq]
  std::vector<double> xyz_in; // geom==2: [3][Ne][Np]
  double R_d, c_vd, R_v, c_vv, T_0, I_v0, grav;
  int sgs;
  double C_s, Pr_t;
  int use_ref;
  std::vector<double> ref_rho, ref_rhoe, ref_rhoq;  // [Ne][Np]
  double shf_bottom;
  int richardson = 0;              // eq. (40) on / off
  double p_0 = 1.0e5;              // reference pressure of theta_v (R25)
  double sponge_alpha = 0.0, sponge_zs = 0.0; int sponge_gamma = 2; double u_relax[3] = {0, 0, 0};   // eq. (A4)-(A5)
  int filter_order = 0; double filter_alpha = 36.0436533891172;   // eq. (52); alpha = -log(2^-52)
  int riemann = 0;                 // 0 Rusanov (eq. 27) | 1 HLLC | 2 Roe
  int metric_form = 0;             // 0 cross-product (R4) | 1 curl-invariant
  int satadj = 0;                  // 1: temperature and condensate from the saturation adjustment of eq. (15)
  double c_vl = 4181.0;            // Table 1
  double p_tr = 611.657, T_tr = 273.16;   // triple point of water (anchor of the saturation vapour pressure, R31)
  double drag_cd = 0.0;            // C_d of the drag law (A2) on the bottom wall, 0 = free slip
  double lhf_bottom = 0.0;         // latent heat flux LHF [W m^-2] added to SHF in the wall energy flux
  double evap_bottom = 0.0;        // evaporation E [kg m^-2 s^-1] into the domain through the bottom wall
  double xi[MAXNQ], w[MAXNQ], D[MAXNQ][MAXNQ];
  double Filt[MAXNQ][MAXNQ];       // 1-D nodal filter matrix V diag(sigma) V^-1
  // optional cache of per-element geometry (same function fills it; see elem_geo)
  bool cached = false;
  std::vector<double> cx, cJa, cJ, cDx;
};

constexpr int NGV = 6;             // gradient variables u, v, w, h_tot, q_t, theta_v
constexpr int NG3 = 3 * NGV;

// ---------------------------------------------------------------- O1: 1-D operators
void legendre(int N, double x, double& P, double& dP) {
  // Bonnet recurrence for P_N and its derivative P_N' (Legendre polynomials).
  double p0 = 1.0, p1 = x, d0 = 0.0, d1 = 1.0;
  if (N == 0) { P = 1.0; dP = 0.0; return; }
  for (int n = 1; n < N; ++n) {
    double p2 = ((2.0 * n + 1.0) * x * p1 - n * p0) / (n + 1.0);
    double d2 = d0 + (2.0 * n + 1.0) * p1;   // P'_{n+1} = P'_{n-1} + (2n+1) P_n
    p0 = p1; p1 = p2; d0 = d1; d1 = d2;
  }
  P = p1; dP = d1;
}

void lgl_nodes_weights(int N, double* xi, double* w) {
  // LGL nodes: -1, +1 and the roots of P_N'(x); Newton on P_N' using the Legendre ODE for P_N''.
  const double pi = 3.14159265358979323846;
  xi[0] = -1.0; xi[N] = 1.0;
  for (int i = 1; i < N; ++i) {
    double x = -std::cos(pi * i / N);
    for (int it = 0; it < 100; ++it) {
      double P, dP; legendre(N, x, P, dP);
      double ddP = (2.0 * x * dP - N * (N + 1.0) * P) / (1.0 - x * x);
      double dx = dP / ddP;
      x -= dx;
      if (std::fabs(dx) < 1e-16) break;
    }
    xi[i] = x;
  }
  for (int i = 0; i <= N / 2; ++i) {  // enforce the exact symmetry of the node set
    double a = 0.5 * (xi[N - i] - xi[i]);
    xi[i] = -a; xi[N - i] = a;
  }
  if (N % 2 == 0) xi[N / 2] = 0.0;
  for (int i = 0; i <= N; ++i) {
    double P, dP; legendre(N, xi[i], P, dP);
    w[i] = 2.0 / (N * (N + 1.0) * P * P);
  }
}

void deriv_matrix(int N, const double* xi, double (*D)[MAXNQ]) {
  // D_ij = L_j'(xi_i) = P_N(xi_i) / (P_N(xi_j) (xi_i - xi_j)), i != j; diagonal = -(sum of the row).
  double PN[MAXNQ];
  for (int i = 0; i <= N; ++i) { double dP; legendre(N, xi[i], PN[i], dP); }
  for (int i = 0; i <= N; ++i) {
    double s = 0.0;
    for (int j = 0; j <= N; ++j) {
      if (i == j) continue;
      D[i][j] = PN[i] / (PN[j] * (xi[i] - xi[j]));
      s += D[i][j];
    }
    D[i][i] = -s;
  }
}

// ---------------------------------------------------------------- O2: mesh and geometry
inline int64_t elem_index(const Ctx& c, int ex, int ey, int ez) {
  return ex + (int64_t)c.ne[0] * (ey + (int64_t)c.ne[1] * ez);
}
inline void elem_coords(const Ctx& c, int64_t e, int& ex, int& ey, int& ez) {
  ex = (int)(e % c.ne[0]); ey = (int)((e / c.ne[0]) % c.ne[1]); ez = (int)(e / ((int64_t)c.ne[0] * c.ne[1]));
}

// Nodal coordinates of element e: x[n][3].  Brick + optional linear-decay warp.
void elem_nodes(const Ctx& c, int64_t e, double* x) {
  const int Nq = c.Nq, Np = c.Np;
  if (c.geom == 2) {
    for (int n = 0; n < Np; ++n)
      for (int d = 0; d < 3; ++d) x[3 * n + d] = c.xyz_in[((int64_t)d * c.Ne + e) * Np + n];
    return;
  }
  int ec[3]; elem_coords(c, e, ec[0], ec[1], ec[2]);
  double h[3];
  for (int d = 0; d < 3; ++d) h[d] = (c.hi[d] - c.lo[d]) / c.ne[d];
  for (int k = 0; k < Nq; ++k)
    for (int j = 0; j < Nq; ++j)
      for (int i = 0; i < Nq; ++i) {
        int n = i + Nq * (j + Nq * k);
        int ijk[3] = {i, j, k};
        double X[3];
        for (int d = 0; d < 3; ++d) X[d] = c.lo[d] + ec[d] * h[d] + 0.5 * (c.xi[ijk[d]] + 1.0) * h[d];
        if (c.geom == 1) {
          // z = ztilde + z_sfc(x,y) * (z_top - ztilde)/(z_top - z_bottom): terrain-following at the
          // bottom, decaying linearly to a flat top (Gal-Chen & Somerville).
          double zs = c.zsfc[(int64_t)(ec[1] * Nq + j) * (c.ne[0] * Nq) + ec[0] * Nq + i];
          X[2] = X[2] + zs * (c.hi[2] - X[2]) / (c.hi[2] - c.lo[2]);
        }
        for (int d = 0; d < 3; ++d) x[3 * n + d] = X[d];
      }
}

// Geometry of one element: x[n][3]; Ja[n][d][cc] = J * d(xi_d)/d(x_cc) (cross-product form); J[n] = det(dx/dxi).
void elem_geo_compute(const Ctx& c, int64_t e, double* x, double* Ja, double* J, double* dxd) {
  const int Nq = c.Nq, Np = c.Np;
  elem_nodes(c, e, x);
  std::vector<double> dX(9 * (size_t)Np);   // dX[n][d][cc] = d x_cc / d xi_d
  for (int k = 0; k < Nq; ++k)
    for (int j = 0; j < Nq; ++j)
      for (int i = 0; i < Nq; ++i) {
        int n = i + Nq * (j + Nq * k);
        double xr[3] = {0, 0, 0}, xs[3] = {0, 0, 0}, xt[3] = {0, 0, 0};  // d(x,y,z)/dxi, /deta, /dzeta
        // The coordinates are differentiated relative to the element's first node: D annihilates constants, so this is
        // eq. (24) unchanged, but the products D_im * x_m no longer carry the element's offset from the origin (up to
        // 3e5 m), whose rounding left spurious off-diagonal metric terms of relative size 8 eps |x| / h ~ 1e-13.
        for (int m = 0; m < Nq; ++m)
          for (int d = 0; d < 3; ++d) {
            xr[d] += c.D[i][m] * (x[3 * (m + Nq * (j + Nq * k)) + d] - x[d]);
            xs[d] += c.D[j][m] * (x[3 * (i + Nq * (m + Nq * k)) + d] - x[d]);
            xt[d] += c.D[k][m] * (x[3 * (i + Nq * (j + Nq * m)) + d] - x[d]);
          }
        for (int d = 0; d < 3; ++d) { dX[9 * n + d] = xr[d]; dX[9 * n + 3 + d] = xs[d]; dX[9 * n + 6 + d] = xt[d]; }
        double* a = Ja + 9 * n;
        // Ja^1 = x_eta x x_zeta ; Ja^2 = x_zeta x x_xi ; Ja^3 = x_xi x x_eta
        a[0] = xs[1] * xt[2] - xs[2] * xt[1]; a[1] = xs[2] * xt[0] - xs[0] * xt[2]; a[2] = xs[0] * xt[1] - xs[1] * xt[0];
        a[3] = xt[1] * xr[2] - xt[2] * xr[1]; a[4] = xt[2] * xr[0] - xt[0] * xr[2]; a[5] = xt[0] * xr[1] - xt[1] * xr[0];
        a[6] = xr[1] * xs[2] - xr[2] * xs[1]; a[7] = xr[2] * xs[0] - xr[0] * xs[2]; a[8] = xr[0] * xs[1] - xr[1] * xs[0];
        J[n] = xr[0] * a[0] + xr[1] * a[1] + xr[2] * a[2];
        dxd[3 * n + 0] = xr[0]; dxd[3 * n + 1] = xs[1]; dxd[3 * n + 2] = xt[2];   // diagonal of dx/dxi: mixing lengths (eq. 39)
      }
  if (c.metric_form == 1) {
    // Curl-invariant form (Kopriva 2006): Ja^i_n = -xhat_i . curl_xi( I_N( X_l grad_xi X_m ) ), (n, m, l) cyclic.  The
    // products are interpolated (taken at the nodes) BEFORE the outer derivative, so sum_i d(Ja^i_n)/d xi_i = 0 holds
    // discretely on any mesh (D_eta D_zeta commute), which the cross-product form only does on extruded meshes (R4).
    std::vector<double> V(3 * (size_t)Np);   // V[n][d] = X_l * d X_m / d xi_d
    for (int nn = 0; nn < 3; ++nn) {
      const int mm = (nn + 1) % 3, ll = (nn + 2) % 3;
      for (int n = 0; n < Np; ++n)
        for (int d = 0; d < 3; ++d) V[3 * n + d] = (x[3 * n + ll] - x[ll]) * dX[9 * n + 3 * d + mm];
      for (int k = 0; k < Nq; ++k)
        for (int j = 0; j < Nq; ++j)
          for (int i = 0; i < Nq; ++i) {
            int n = i + Nq * (j + Nq * k);
            double dV[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};   // dV[a][d] = d V_d / d xi_a
            for (int m = 0; m < Nq; ++m)
              for (int d = 0; d < 3; ++d) {
                dV[0][d] += c.D[i][m] * V[3 * (m + Nq * (j + Nq * k)) + d];
                dV[1][d] += c.D[j][m] * V[3 * (i + Nq * (m + Nq * k)) + d];
                dV[2][d] += c.D[k][m] * V[3 * (i + Nq * (j + Nq * m)) + d];
              }
            // curl components: (d_eta V_3 - d_zeta V_2, d_zeta V_1 - d_xi V_3, d_xi V_2 - d_eta V_1)
            Ja[9 * n + 0 + nn] = -(dV[1][2] - dV[2][1]);
            Ja[9 * n + 3 + nn] = -(dV[2][0] - dV[0][2]);
            Ja[9 * n + 6 + nn] = -(dV[0][1] - dV[1][0]);
          }
    }
  }
}

struct Geo {  // views for one element
  const double *x, *Ja, *J, *dxd;
  std::vector<double> sx, sJa, sJ, sDx;
};
void elem_geo(const Ctx& c, int64_t e, Geo& g) {
  const int Np = c.Np;
  if (c.cached) {
    g.x = &c.cx[(size_t)e * Np * 3]; g.Ja = &c.cJa[(size_t)e * Np * 9]; g.J = &c.cJ[(size_t)e * Np];
    g.dxd = &c.cDx[(size_t)e * Np * 3];
    return;
  }
  g.sx.resize(3 * Np); g.sJa.resize(9 * Np); g.sJ.resize(Np); g.sDx.resize(3 * Np);
  elem_geo_compute(c, e, g.sx.data(), g.sJa.data(), g.sJ.data(), g.sDx.data());
  g.x = g.sx.data(); g.Ja = g.sJa.data(); g.J = g.sJ.data(); g.dxd = g.sDx.data();
}

// neighbour across face f (0..5 = -xi,+xi,-eta,+eta,-zeta,+zeta); -1 if the face is a wall.
int64_t neighbour(const Ctx& c, int64_t e, int f) {
  int ec[3]; elem_coords(c, e, ec[0], ec[1], ec[2]);
  int d = f / 2, s = (f % 2) ? +1 : -1;
  int v = ec[d] + s;
  if (v < 0 || v >= c.ne[d]) {
    if (c.bc[d] != 0) return -1;
    v = (v + c.ne[d]) % c.ne[d];
  }
  ec[d] = v;
  return elem_index(c, ec[0], ec[1], ec[2]);
}

// node of element at face f with in-face indices (a,b); and the coincident node seen from the neighbour.
inline int face_node(int Nq, int f, int a, int b, bool other_side) {
  int d = f / 2;
  int at = (f % 2) ? (Nq - 1) : 0;
  if (other_side) at = (Nq - 1) - at;
  int i, j, k;
  if (d == 0) { i = at; j = a; k = b; }
  else if (d == 1) { i = a; j = at; k = b; }
  else { i = a; j = b; k = at; }
  return i + Nq * (j + Nq * k);
}

// ---------------------------------------------------------------- O3: thermodynamics at a node
struct Prim {
  double rho, u[3], q, K, Phi, T, p, pp /* p - p_r */, htot, c, rho_r, theta_v, ql /* liquid specific humidity */;
};

// O15.  Saturation vapour pressure over liquid with constant heat capacities (Romps 2008): Clausius-Clapeyron
//   d ln p* / dT = L(T) / (R_v T^2),  L(T) = L_v0 + (c_pv - c_pl)(T - T_0),  c_pv = c_vv + R_v,  c_pl = c_vl,
// integrated from the triple point (T_tr, p_tr):
//   p*(T) = p_tr (T / T_tr)^(dcp / R_v) exp[ ((L_v0 - dcp T_0) / R_v) (1 / T_tr - 1 / T) ],  dcp = c_pv - c_pl.
double sat_vapor_pressure(const Ctx& c, double T) {
  double dcp = (c.c_vv + c.R_v) - c.c_vl, Lv0 = c.I_v0 + c.R_v * c.T_0;        // eq. (9)
  return c.p_tr * std::pow(T / c.T_tr, dcp / c.R_v) * std::exp((Lv0 - dcp * c.T_0) / c.R_v * (1.0 / c.T_tr - 1.0 / T));
}
// saturation specific humidity at given density: q_v* = p*(T) / (rho R_v T)
double sat_q(const Ctx& c, double T, double rho) { return sat_vapor_pressure(c, T) / (rho * c.R_v * T); }

// internal energy at equilibrium I*(T; rho, q_t) of eq. (15) with eq. (7)-(8): unsaturated (q_v = q_t) or saturated with
// the excess q_t - q_v*(T, rho) as liquid
double internal_energy_eq(const Ctx& c, double T, double rho, double qt, double* ql_out) {
  double qvs = sat_q(c, T, rho);
  double qv = std::min(qt, qvs), ql = qt - qv;
  if (ql_out) *ql_out = ql;
  return (1.0 - qt) * c.c_vd * (T - c.T_0) + qv * (c.c_vv * (T - c.T_0) + c.I_v0) + ql * c.c_vl * (T - c.T_0);
}

// root T of I*(T; rho, q_t) - I = 0 (eq. 15) by Newton iterations with the analytical derivative; ql = condensate
double saturation_adjustment(const Ctx& c, double I, double rho, double qt, double* ql) {
  double cvm = c.c_vd * (1.0 - qt) + c.c_vv * qt;
  double T = c.T_0 + (I - qt * c.I_v0) / cvm;                 // unsaturated: eq. (7)-(8) solved for T
  if (qt <= sat_q(c, T, rho)) { *ql = 0.0; return T; }
  double dcp = (c.c_vv + c.R_v) - c.c_vl, Lv0 = c.I_v0 + c.R_v * c.T_0;
  for (int it = 0; it < 50; ++it) {
    double qvs = sat_q(c, T, rho);
    double f = (1.0 - qt) * c.c_vd * (T - c.T_0) + qvs * (c.c_vv * (T - c.T_0) + c.I_v0) + (qt - qvs) * c.c_vl * (T - c.T_0) - I;
    double L = Lv0 + dcp * (T - c.T_0);
    double dqvs = qvs * (L / (c.R_v * T * T) - 1.0 / T);      // d q_v* / dT at fixed rho
    double df = (1.0 - qt) * c.c_vd + qvs * c.c_vv + (qt - qvs) * c.c_vl + dqvs * ((c.c_vv - c.c_vl) * (T - c.T_0) + c.I_v0);
    double dT = f / df;
    T -= dT;
    if (std::fabs(dT) <= 1e-14 * T) break;
  }
  *ql = qt - sat_q(c, T, rho);
  return T;
}

Prim primitives(const Ctx& c, const double* Y, double z, bool has_ref, double rr, double rer, double rqr) {
  Prim P;
  P.rho = Y[0];
  for (int d = 0; d < 3; ++d) P.u[d] = Y[1 + d] / Y[0];
  P.q = (c.nvar == 6) ? Y[5] / Y[0] : 0.0;
  P.Phi = c.grav * z;                                                   // Phi = g z
  P.K = 0.5 * (Y[1] * Y[1] + Y[2] * Y[2] + Y[3] * Y[3]) / Y[0];          // rho |u|^2 / 2
  double eint = Y[4] / Y[0] - 0.5 * (P.u[0] * P.u[0] + P.u[1] * P.u[1] + P.u[2] * P.u[2]) - P.Phi;  // eq. (6)
  double cvm = c.c_vd * (1.0 - P.q) + c.c_vv * P.q;                     // eq. (7)-(8), q_v=q_t, q_l=q_i=0
  double Rm = c.R_d * (1.0 - P.q) + c.R_v * P.q;                        // eq. (14)
  P.T = c.T_0 + (eint - P.q * c.I_v0) / cvm;
  P.ql = 0.0;
  if (c.satadj && c.nvar == 6) {
    P.T = saturation_adjustment(c, eint, P.rho, P.q, &P.ql);            // eq. (15)
    cvm = c.c_vd * (1.0 - P.q) + c.c_vv * (P.q - P.ql) + c.c_vl * P.ql;   // eq. (7)-(8) with condensate
    Rm = c.R_d * (1.0 - P.q) + c.R_v * (P.q - P.ql);                    // eq. (14): R_d [1 + (eps - 1) q_t - eps q_c]
  }
  P.p = P.rho * Rm * P.T;                                               // eq. (13)
  P.htot = Y[4] / Y[0] + Rm * P.T;                                      // (rho e + p)/rho
  P.c = std::sqrt((1.0 + Rm / cvm) * Rm * P.T);
  // virtual potential temperature without condensate (R25): theta_v = T (R_m / R_d) (p_0 / p)^(R_d / c_pd)
  P.theta_v = P.T * (Rm / c.R_d) * std::pow(c.p_0 / P.p, c.R_d / (c.c_vd + c.R_d));
  P.rho_r = 0.0;
  if (has_ref && c.satadj && c.nvar == 6) {
    // with condensate the pressure is no longer linear in the state (R12 does not apply): p_r is the pressure of the
    // resting reference state under the same equation of state, and p' the plain difference
    double Yr[6] = {rr, 0.0, 0.0, 0.0, rer, rqr};
    Prim Pr = primitives(c, Yr, z, false, 0, 0, 0);
    P.pp = P.p - Pr.p;
    P.rho_r = rr;
  } else if (has_ref) {
    // R12: p - p_r evaluated from state differences (exact identity for the EOS above, with
    // p_r := EOS pressure of the resting reference state (rho_r, 0, rhoe_r, rhoq_r)).
    double rq = (c.nvar == 6) ? Y[5] : 0.0;
    double a = c.R_v - c.R_d, b = c.c_vv - c.c_vd;
    double qr = rqr / rr;
    double cvmr = c.c_vd * (1.0 - qr) + c.c_vv * qr;
    double kappa = Rm / cvm;
    double dE = (Y[4] - rer) - (Y[0] - rr) * P.Phi - (rq - rqr) * c.I_v0;
    double Er = rer - rr * P.Phi - rqr * c.I_v0;
    double dkappa = (P.q - qr) * (a * c.c_vd - c.R_d * b) / (cvm * cvmr);
    P.pp = kappa * dE - kappa * P.K + dkappa * Er + c.T_0 * (c.R_d * (Y[0] - rr) + a * (rq - rqr));
    P.rho_r = rr;
  } else {
    P.pp = P.p;
  }
  return P;
}

inline Prim prim_at(const Ctx& c, const double* Q, int64_t e, int n, double z) {
  const double* Y = Q + ((size_t)e * c.Np + n) * c.nvar;
  if (c.use_ref) {
    size_t id = (size_t)e * c.Np + n;
    return primitives(c, Y, z, true, c.ref_rho[id], c.ref_rhoe[id], (c.nvar == 6) ? c.ref_rhoq[id] : 0.0);
  }
  return primitives(c, Y, z, false, 0, 0, 0);
}

// gradient variables s = (u, v, w, h_tot, q_t, theta_v)   (eq. 33, 35, 37, 40)
inline void grad_vars(const Prim& P, double* s) {
  s[0] = P.u[0]; s[1] = P.u[1]; s[2] = P.u[2]; s[3] = P.htot; s[4] = P.q; s[5] = P.theta_v;
}

// ---------------------------------------------------------------- O4: BR1 gradient of one element
// G[n][s][cc] = d s / d x_cc, s = u,v,w,h_tot,q  (15 values per node)
void gradient_element(const Ctx& c, const double* Q, int64_t e, double* G) {
  const int Nq = c.Nq, Np = c.Np;
  Geo g; elem_geo(c, e, g);
  std::vector<double> s(NGV * Np);
  for (int n = 0; n < Np; ++n) {
    Prim P = prim_at(c, Q, e, n, g.x[3 * n + 2]);
    grad_vars(P, &s[NGV * n]);
  }
  // volume part: G_cc = sum_d (Ja^d_cc / J) (D_d s)      (eq. 24, 28)
  for (int k = 0; k < Nq; ++k)
    for (int j = 0; j < Nq; ++j)
      for (int i = 0; i < Nq; ++i) {
        int n = i + Nq * (j + Nq * k);
        for (int v = 0; v < NGV; ++v) {
          double dr = 0, ds = 0, dt = 0;
          for (int m = 0; m < Nq; ++m) {
            dr += c.D[i][m] * s[NGV * (m + Nq * (j + Nq * k)) + v];
            ds += c.D[j][m] * s[NGV * (i + Nq * (m + Nq * k)) + v];
            dt += c.D[k][m] * s[NGV * (i + Nq * (j + Nq * m)) + v];
          }
          const double* a = g.Ja + 9 * n;
          for (int cc = 0; cc < 3; ++cc)
            G[(n * NGV + v) * 3 + cc] = (a[0 + cc] * dr + a[3 + cc] * ds + a[6 + cc] * dt) / g.J[n];
        }
      }
  // surface part: + (sJ/(w_0 J)) n_cc (s* - s^-)            (eq. 30 with central s*)
  for (int f = 0; f < 6; ++f) {
    int64_t en = neighbour(c, e, f);
    int d = f / 2; double sgn = (f % 2) ? 1.0 : -1.0;
    Geo gn; if (en >= 0) elem_geo(c, en, gn);
    for (int b = 0; b < Nq; ++b)
      for (int a_ = 0; a_ < Nq; ++a_) {
        int n = face_node(Nq, f, a_, b, false);
        const double* Ja = g.Ja + 9 * n + 3 * d;
        double sJ = std::sqrt(Ja[0] * Ja[0] + Ja[1] * Ja[1] + Ja[2] * Ja[2]);
        double nrm[3] = {sgn * Ja[0] / sJ, sgn * Ja[1] / sJ, sgn * Ja[2] / sJ};
        double lift = sJ / (c.w[0] * g.J[n]);
        double sm[NGV], sstar[NGV];
        for (int v = 0; v < NGV; ++v) sm[v] = s[NGV * n + v];
        if (en >= 0) {
          int nn = face_node(Nq, f, a_, b, true);
          Prim Pp = prim_at(c, Q, en, nn, gn.x[3 * nn + 2]);
          double sp[NGV]; grad_vars(Pp, sp);
          for (int v = 0; v < NGV; ++v) sstar[v] = 0.5 * (sm[v] + sp[v]);
        } else {
          // wall: u_bc = u^- - (n.u^-) n (A6); scalars chi_bc = chi^- (homogeneous Neumann, A8)
          double un = sm[0] * nrm[0] + sm[1] * nrm[1] + sm[2] * nrm[2];
          for (int v = 0; v < 3; ++v) sstar[v] = sm[v] - un * nrm[v];
          sstar[3] = sm[3]; sstar[4] = sm[4]; sstar[5] = sm[5];
        }
        for (int v = 0; v < NGV; ++v)
          for (int cc = 0; cc < 3; ++cc) G[(n * NGV + v) * 3 + cc] += lift * nrm[cc] * (sstar[v] - sm[v]);
      }
  }
}

// ---------------------------------------------------------------- O5/O6: fluxes at a node
// F[v][cc]: physical flux of variable v in direction cc.
void flux_first_order(const Ctx& c, const double* Y, const Prim& P, double (*F)[3]) {
  for (int cc = 0; cc < 3; ++cc) {
    F[0][cc] = Y[1 + cc];                                   // rho u            eq. (1)
    for (int i = 0; i < 3; ++i) F[1 + i][cc] = Y[1 + i] * P.u[cc] + ((i == cc) ? P.pp : 0.0);  // eq. (4)
    F[4][cc] = (Y[4] + P.p) * P.u[cc];                      // (rho e + p) u    eq. (5)
    if (c.nvar == 6) F[5][cc] = Y[5] * P.u[cc];             // rho q u          eq. (2)
  }
}

// Eddy viscosity at a node.  G[s][cc] = d s / d x_cc for s = u, v, w, h_tot, q, theta_v; dxd = diagonal of dx/dxi.
//   sgs = 1  Smagorinsky-Lilly (eq. 38) with Delta = (8 J)^(1/3) / N (R7)
//   sgs = 2  Vreman (eq. 39a-d) with the mixing lengths Delta_m = 2 |d x_m / d xi_m| / N (= L_m / N on bricks; R24)
//   richardson: nu_t is multiplied by f_b of eq. (40), Ri = (g / theta_v) (d theta_v / dz) / |S|^2, |S|^2 = 2 S_ij S_ij
double eddy_viscosity(const Ctx& c, const double* G, double J, const double* dxd, double theta_v) {
  double S[3][3];
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) S[i][j] = 0.5 * (G[i * 3 + j] + G[j * 3 + i]);   // eq. (33); G[s][cc]=d u_s/d x_cc
  double ss = 0;
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) ss += S[i][j] * S[i][j];
  double nu;
  if (c.sgs == 2) {
    double beta[3][3], aa = 0;
    for (int i = 0; i < 3; ++i)
      for (int j = 0; j < 3; ++j) {
        double b = 0;
        for (int m = 0; m < 3; ++m) {
          double Dm = 2.0 * std::fabs(dxd[m]) / c.N;
          b += Dm * Dm * G[i * 3 + m] * G[j * 3 + m];                              // eq. (39c)
        }
        beta[i][j] = b;
        aa += G[i * 3 + j] * G[i * 3 + j];                                         // u_ij u_ij
      }
    double B = beta[0][0] * beta[1][1] + beta[0][0] * beta[2][2] + beta[1][1] * beta[2][2] -
               (beta[0][2] * beta[0][2] + beta[0][1] * beta[0][1] + beta[1][2] * beta[1][2]);   // eq. (39b)
    nu = (aa > 0.0 && B > 0.0) ? 2.5 * c.C_s * c.C_s * std::sqrt(B / aa) : 0.0;    // eq. (39a); 0/0 := 0 (no flow, no mixing)
  } else {
    double Delta = std::cbrt(8.0 * J) / c.N;
    nu = (c.C_s * Delta) * (c.C_s * Delta) * std::sqrt(2.0 * ss);
  }
  if (c.richardson) {
    double N2 = (c.grav / theta_v) * G[5 * 3 + 2];
    double fb = 1.0;                                                               // Ri <= 0
    if (N2 > 0.0) {
      double Ri = N2 / (2.0 * ss);                                                 // |S|^2 = 0: Ri = inf, f_b = 0
      double t = 1.0 - Ri / c.Pr_t;
      fb = (t > 0.0) ? std::sqrt(std::sqrt(t)) : 0.0;                               // eq. (40)
    }
    nu *= fb;
  }
  return nu;
}

void flux_second_order(const Ctx& c, const double* Y, const Prim& P, const double* G, double J, const double* dxd,
                       double (*F)[3]) {
  double nu = eddy_viscosity(c, G, J, dxd, P.theta_v);
  double Dt = nu / c.Pr_t;                                   // eq. (36)
  double tau[3][3];
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) tau[i][j] = -2.0 * nu * 0.5 * (G[i * 3 + j] + G[j * 3 + i]);  // eq. (34)
  for (int cc = 0; cc < 3; ++cc) {
    double dq = (c.nvar == 6) ? -Dt * G[4 * 3 + cc] : 0.0;   // eq. (35)
    double JD = -Dt * G[3 * 3 + cc];                         // eq. (37)
    F[0][cc] = (c.nvar == 6) ? P.rho * dq : 0.0;             // eq. (1)-(2): mass carries the water diffusion
    for (int i = 0; i < 3; ++i) F[1 + i][cc] = P.rho * tau[i][cc] + dq * Y[1 + i];   // eq. (4)
    F[4][cc] = P.rho * (tau[cc][0] * P.u[0] + tau[cc][1] * P.u[1] + tau[cc][2] * P.u[2]) + P.rho * JD;  // eq. (5)
    if (c.nvar == 6) F[5][cc] = P.rho * dq;
  }
}

// ---------------------------------------------------------------- O8: numerical flux n.F1* of two states
// riemann = 0: Rusanov (eq. 27 with R1, R2).  riemann = 1: HLLC (named at P:L256; Toro, Spruce & Speares 1994) with the
// wave-speed estimates S_L = min(u_L - c_L, u_R - c_R), S_R = max(u_L + c_L, u_R + c_R); the momentum flux carries
// p' = p - p_r (the reference pressure is the same on both sides of a face), the energy flux the full p; rho q is
// advected with the mass flux.  L = "-" side, R = "+" side, velocities along the outward normal n.
void numerical_flux(const Ctx& c, const double* Ym, const Prim& Pm, const double (*F1m)[3], const double* Yp, const Prim& Pp,
                    const double (*F1p)[3], const double* nrm, double* Fstar) {
  const int nv = c.nvar;
  double unm = Pm.u[0] * nrm[0] + Pm.u[1] * nrm[1] + Pm.u[2] * nrm[2];
  double unp = Pp.u[0] * nrm[0] + Pp.u[1] * nrm[1] + Pp.u[2] * nrm[2];
  double nFm[6], nFp[6];
  for (int v = 0; v < nv; ++v) {
    nFm[v] = 0; nFp[v] = 0;
    for (int cc = 0; cc < 3; ++cc) { nFm[v] += nrm[cc] * F1m[v][cc]; nFp[v] += nrm[cc] * F1p[v][cc]; }
  }
  if (c.riemann == 0) {
    double lam = std::max(std::fabs(unm) + Pm.c, std::fabs(unp) + Pp.c);   // R2
    for (int v = 0; v < nv; ++v) Fstar[v] = 0.5 * (nFm[v] + nFp[v]) + 0.5 * lam * (Ym[v] - Yp[v]);   // eq. (27), reading R1
    return;
  }
  if (c.riemann == 2) {
    // Roe (named at P:L256; Roe 1981, textbook form): F* = (1/2)(F^- + F^+) - (1/2) sum_k |lambda_k| alpha_k r_k with the
    // sqrt(rho)-weighted averages u~, H~ (total enthalpy), q~.  With the mixture frozen at q~ the EOS of eq. (6)-(14) is an
    // ideal gas with gamma - 1 = kappa~ = R_m / c_vm and the energy shifted by s~ = Phi + q~ I_v0 - c_vm T_0:
    // p = kappa (rho e - rho |u|^2 / 2 - rho s), hence c~^2 = kappa~ (H~ - s~ - |u~|^2 / 2).  Exact Roe linearisation for dry
    // air; rho q is a passive wave of speed u~_n (reading R32).  No entropy fix.
    double wm = std::sqrt(Ym[0]), wp = std::sqrt(Yp[0]), iw = 1.0 / (wm + wp);
    double ut[3], un = 0, K = 0;
    for (int i = 0; i < 3; ++i) { ut[i] = (wm * Pm.u[i] + wp * Pp.u[i]) * iw; un += ut[i] * nrm[i]; K += 0.5 * ut[i] * ut[i]; }
    double H = (wm * Pm.htot + wp * Pp.htot) * iw;
    double q = (nv == 6) ? (wm * Pm.q + wp * Pp.q) * iw : 0.0;
    double cvm = c.c_vd * (1.0 - q) + c.c_vv * q, Rm = c.R_d * (1.0 - q) + c.R_v * q;
    double kappa = Rm / cvm;
    double sh = Pm.Phi + q * c.I_v0 - cvm * c.T_0;          // Phi is the same on both sides of a face
    double c2 = kappa * (H - sh - K), cs = std::sqrt(c2);
    double rt = wm * wp;                                     // rho~
    double drho = Yp[0] - Ym[0], dp = Pp.pp - Pm.pp, dun = unp - unm;
    double du[3]; for (int i = 0; i < 3; ++i) du[i] = Pp.u[i] - Pm.u[i];
    double a1 = (dp - rt * cs * dun) / (2.0 * c2), a5 = (dp + rt * cs * dun) / (2.0 * c2), a2 = drho - dp / c2;
    double l1 = std::fabs(un - cs), l2 = std::fabs(un), l5 = std::fabs(un + cs);
    double D[6];
    D[0] = l1 * a1 + l2 * a2 + l5 * a5;
    double udu = 0;
    for (int i = 0; i < 3; ++i) {
      double sh_i = du[i] - dun * nrm[i];                    // shear part of the velocity jump
      D[1 + i] = l1 * a1 * (ut[i] - cs * nrm[i]) + l2 * (a2 * ut[i] + rt * sh_i) + l5 * a5 * (ut[i] + cs * nrm[i]);
      udu += ut[i] * sh_i;
    }
    D[4] = l1 * a1 * (H - cs * un) + l2 * (a2 * (K + sh) + rt * udu) + l5 * a5 * (H + cs * un);
    if (nv == 6) D[5] = (l1 * a1 + l2 * a2 + l5 * a5) * q + l2 * rt * (Pp.q - Pm.q);
    for (int v = 0; v < nv; ++v) Fstar[v] = 0.5 * (nFm[v] + nFp[v]) - 0.5 * D[v];
    return;
  }
  double SL = std::min(unm - Pm.c, unp - Pp.c), SR = std::max(unm + Pm.c, unp + Pp.c);
  double Sstar = ((Pp.pp - Pm.pp) + Ym[0] * unm * (SL - unm) - Yp[0] * unp * (SR - unp)) /
                 (Ym[0] * (SL - unm) - Yp[0] * (SR - unp));
  if (SL >= 0.0) { for (int v = 0; v < nv; ++v) Fstar[v] = nFm[v]; return; }
  if (SR <= 0.0) { for (int v = 0; v < nv; ++v) Fstar[v] = nFp[v]; return; }
  const bool left = Sstar >= 0.0;
  const double* Y = left ? Ym : Yp; const Prim& P = left ? Pm : Pp;
  const double un = left ? unm : unp, SK = left ? SL : SR;
  const double* nF = left ? nFm : nFp;
  // F* = F_K + S_K (U*_K - U_K) with U*_K = rho*_K [1; u + (S* - u_n) n; E/rho + (S* - u_n)(S* + p / (rho (S_K - u_n))); q],
  // rho*_K = rho (S_K - u_n) / (S_K - S*).  The jump U*_K - U_K is formed analytically (rho* - rho = rho (S* - u_n) /
  // (S_K - S*)): multiplying the rounded difference of two O(rho c) numbers by S_K would leave an error of one ulp of
  // rho c in every flux, which is 1e-10 of the tendency of a flow near rest.
  double ds = Sstar - un;
  double rs = Y[0] * (SK - un) / (SK - Sstar);            // rho*_K
  double drho = Y[0] * ds / (SK - Sstar);                 // rho*_K - rho_K
  double dU[6];
  dU[0] = drho;
  for (int i = 0; i < 3; ++i) dU[1 + i] = drho * P.u[i] + rs * ds * nrm[i];
  dU[4] = drho * (Y[4] / Y[0]) + rs * ds * (Sstar + P.p / (Y[0] * (SK - un)));
  if (nv == 6) dU[5] = drho * P.q;
  for (int v = 0; v < nv; ++v) Fstar[v] = nF[v] + SK * dU[v];
}

// ---------------------------------------------------------------- O7/O8: tendency of one element
// Ge = gradient of this element [Np][18]; Gn[f] = gradient array of the neighbour across face f (or null).
// form: 0 weak (eq. 26), 1 strong (eq. 32).
void rhs_element(const Ctx& c, const double* Q, int64_t e, const double* Ge, const double* const* Gn, int form,
                 double* dQ) {
  const int Nq = c.Nq, Np = c.Np, nv = c.nvar;
  Geo g; elem_geo(c, e, g);
  std::vector<Prim> P(Np);
  std::vector<double> Ft((size_t)Np * nv * 3);   // contravariant fluxes Ft[n][v][d] = Ja^d . F
  std::vector<double> Fp((size_t)Np * nv * 3);   // physical fluxes     Fp[n][v][cc]
  for (int n = 0; n < Np; ++n) {
    const double* Y = Q + ((size_t)e * Np + n) * nv;
    P[n] = prim_at(c, Q, e, n, g.x[3 * n + 2]);
    double F1[6][3], F2[6][3];
    flux_first_order(c, Y, P[n], F1);
    if (c.sgs) flux_second_order(c, Y, P[n], Ge + NG3 * n, g.J[n], g.dxd + 3 * n, F2);
    const double* a = g.Ja + 9 * n;
    for (int v = 0; v < nv; ++v) {
      double F[3];
      for (int cc = 0; cc < 3; ++cc) F[cc] = F1[v][cc] + (c.sgs ? F2[v][cc] : 0.0);
      for (int cc = 0; cc < 3; ++cc) Fp[((size_t)n * nv + v) * 3 + cc] = F[cc];
      for (int d = 0; d < 3; ++d) Ft[((size_t)n * nv + v) * 3 + d] = a[3 * d] * F[0] + a[3 * d + 1] * F[1] + a[3 * d + 2] * F[2];
    }
  }
  // volume term + source
  for (int k = 0; k < Nq; ++k)
    for (int j = 0; j < Nq; ++j)
      for (int i = 0; i < Nq; ++i) {
        int n = i + Nq * (j + Nq * k);
        for (int v = 0; v < nv; ++v) {
          double acc = 0;
          if (form == 0) {
            // weak: (1/J) [ (1/w_i) sum_m D_mi w_m Ft^1(m,j,k) + ... ]   (eq. 26, LGL quadrature)
            double a1 = 0, a2 = 0, a3 = 0;
            for (int m = 0; m < Nq; ++m) {
              a1 += c.D[m][i] * c.w[m] * Ft[((size_t)(m + Nq * (j + Nq * k)) * nv + v) * 3 + 0];
              a2 += c.D[m][j] * c.w[m] * Ft[((size_t)(i + Nq * (m + Nq * k)) * nv + v) * 3 + 1];
              a3 += c.D[m][k] * c.w[m] * Ft[((size_t)(i + Nq * (j + Nq * m)) * nv + v) * 3 + 2];
            }
            acc = (a1 / c.w[i] + a2 / c.w[j] + a3 / c.w[k]) / g.J[n];
          } else {
            // strong: -(1/J) sum_d D_d Ft^d                               (eq. 32)
            double a1 = 0, a2 = 0, a3 = 0;
            for (int m = 0; m < Nq; ++m) {
              a1 += c.D[i][m] * Ft[((size_t)(m + Nq * (j + Nq * k)) * nv + v) * 3 + 0];
              a2 += c.D[j][m] * Ft[((size_t)(i + Nq * (m + Nq * k)) * nv + v) * 3 + 1];
              a3 += c.D[k][m] * Ft[((size_t)(i + Nq * (j + Nq * m)) * nv + v) * 3 + 2];
            }
            acc = -(a1 + a2 + a3) / g.J[n];
          }
          dQ[(size_t)n * nv + v] = acc;
        }
        // source: -(rho - rho_r) grad Phi, grad Phi = g zhat          (eq. 4)
        dQ[(size_t)n * nv + 3] += -(P[n].rho - P[n].rho_r) * c.grav;
        // Rayleigh sponge (A4)-(A5) with reading R18 (the pi that (A5) lacks): tau_s = alpha sin^gamma(pi/2 (z-z_s)/(z_top-z_s))
        double z = g.x[3 * n + 2];
        if (c.sponge_alpha > 0.0 && z > c.sponge_zs) {
          const double pi = 3.14159265358979323846;
          double tau = c.sponge_alpha * std::pow(std::sin(0.5 * pi * (z - c.sponge_zs) / (c.hi[2] - c.sponge_zs)), c.sponge_gamma);
          const double* Y = Q + ((size_t)e * Np + n) * nv;
          for (int i = 0; i < 3; ++i) dQ[(size_t)n * nv + 1 + i] -= tau * (Y[1 + i] - Y[0] * c.u_relax[i]);
        }
      }
  // surface term
  for (int f = 0; f < 6; ++f) {
    int64_t en = neighbour(c, e, f);
    int d = f / 2; double sgn = (f % 2) ? 1.0 : -1.0;
    Geo gn; if (en >= 0) elem_geo(c, en, gn);
    for (int b = 0; b < Nq; ++b)
      for (int a_ = 0; a_ < Nq; ++a_) {
        int n = face_node(Nq, f, a_, b, false);
        const double* Ja = g.Ja + 9 * n + 3 * d;
        double sJ = std::sqrt(Ja[0] * Ja[0] + Ja[1] * Ja[1] + Ja[2] * Ja[2]);
        double nrm[3] = {sgn * Ja[0] / sJ, sgn * Ja[1] / sJ, sgn * Ja[2] / sJ};
        double lift = sJ / (c.w[0] * g.J[n]);
        const double* Ym = Q + ((size_t)e * Np + n) * nv;
        const Prim& Pm = P[n];
        double F1m[6][3]; flux_first_order(c, Ym, Pm, F1m);
        double F2m[6][3];
        if (c.sgs) flux_second_order(c, Ym, Pm, Ge + NG3 * n, g.J[n], g.dxd + 3 * n, F2m);
        double Yp[6]; Prim Pp; double F1p[6][3], F2p[6][3];
        double Fstar[6];
        if (en >= 0) {
          int nn = face_node(Nq, f, a_, b, true);
          const double* Yn = Q + ((size_t)en * Np + nn) * nv;
          for (int v = 0; v < nv; ++v) Yp[v] = Yn[v];
          Pp = prim_at(c, Q, en, nn, gn.x[3 * nn + 2]);
          flux_first_order(c, Yp, Pp, F1p);
          if (c.sgs) flux_second_order(c, Yp, Pp, Gn[f] + NG3 * nn, gn.J[nn], gn.dxd + 3 * nn, F2p);
        } else {
          // wall ghost state: mirror the normal momentum (A6)-(A7); scalars copied (A8); p_r^+ = p_r^-
          double mn = Ym[1] * nrm[0] + Ym[2] * nrm[1] + Ym[3] * nrm[2];
          Yp[0] = Ym[0]; Yp[4] = Ym[4]; if (nv == 6) Yp[5] = Ym[5];
          for (int i = 0; i < 3; ++i) Yp[1 + i] = Ym[1 + i] - 2.0 * mn * nrm[i];
          Pp = Pm;
          for (int i = 0; i < 3; ++i) Pp.u[i] = Yp[1 + i] / Yp[0];
          flux_first_order(c, Yp, Pp, F1p);
        }
        numerical_flux(c, Ym, Pm, F1m, Yp, Pp, F1p, nrm, Fstar);               // eq. (27) / HLLC
        if (c.sgs && en >= 0)
          for (int v = 0; v < nv; ++v) {
            double a2 = 0;
            for (int cc = 0; cc < 3; ++cc) a2 += nrm[cc] * 0.5 * (F2m[v][cc] + F2p[v][cc]);   // P:L274, R6
            Fstar[v] += a2;
          }  // wall: n.F2* = 0 (R10)
        if (en < 0 && f == 4 && c.shf_bottom != 0.0) Fstar[4] += -c.shf_bottom;  // prescribed upward energy flux
        if (en < 0 && f == 4) {
          // O14 (R30).  n_in = -nrm is the inward normal of App. A.  All are fluxes INTO the domain, Fstar is outward.
          // energy: n_in . rho (J + D) = SHF + LHF; water and, with it, mass (same right-hand side):
          // E = n_in . (rho d_qv)
          Fstar[4] += -c.lhf_bottom;
          if (nv == 6) { Fstar[5] += -c.evap_bottom; Fstar[0] += -c.evap_bottom; }
          if (c.drag_cd > 0.0) {
            // drag law (A2): n_in . (rho tau) = -rho C_d |u_p,int| u_p,int, u_p,int = wall-parallel velocity at the first
            // layer of interior nodes of the surface-adjacent element: the node above this one in the column
            int ni = n + Nq * Nq;
            Prim Pi = prim_at(c, Q, e, ni, g.x[3 * ni + 2]);
            double un = Pi.u[0] * nrm[0] + Pi.u[1] * nrm[1] + Pi.u[2] * nrm[2];
            double up[3], mag = 0;
            for (int i = 0; i < 3; ++i) { up[i] = Pi.u[i] - un * nrm[i]; mag += up[i] * up[i]; }
            mag = std::sqrt(mag);
            // momentum equation: -div(rho tau); outward normal flux nrm . (rho tau) = -n_in . (rho tau)
            for (int i = 0; i < 3; ++i) Fstar[1 + i] += Ym[0] * c.drag_cd * mag * up[i];
          }
        }
        for (int v = 0; v < nv; ++v) {
          if (form == 0) {
            dQ[(size_t)n * nv + v] -= lift * Fstar[v];
          } else {
            double nF = 0;
            for (int cc = 0; cc < 3; ++cc) nF += nrm[cc] * Fp[((size_t)n * nv + v) * 3 + cc];
            dQ[(size_t)n * nv + v] += lift * (nF - Fstar[v]);
          }
        }
      }
  }
}

void gradient_all(const Ctx& c, const double* Q, double* G) {
#pragma omp parallel for schedule(static)
  for (int64_t e = 0; e < c.Ne; ++e) gradient_element(c, Q, e, G + (size_t)e * c.Np * NG3);
}

void rhs_all(const Ctx& c, const double* Q, double* dQ, int form) {
  std::vector<double> G;
  if (c.sgs) { G.resize((size_t)c.Ne * c.Np * NG3); gradient_all(c, Q, G.data()); }
#pragma omp parallel for schedule(static)
  for (int64_t e = 0; e < c.Ne; ++e) {
    const double* Gn[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    const double* Ge = nullptr;
    if (c.sgs) {
      Ge = &G[(size_t)e * c.Np * NG3];
      for (int f = 0; f < 6; ++f) { int64_t en = neighbour(c, e, f); if (en >= 0) Gn[f] = &G[(size_t)en * c.Np * NG3]; }
    }
    rhs_element(c, Q, e, Ge, Gn, form, dQ + (size_t)e * c.Np * c.nvar);
  }
}

// LSRK54 coefficients, Carpenter & Kennedy (1994), 2N-storage (5,4) scheme.
const double RKA[5] = {0.0, -567301805773.0 / 1357537059087.0, -2404267990393.0 / 2016746695238.0,
                       -3550918686646.0 / 2091501179385.0, -1275806237668.0 / 842570457699.0};
const double RKB[5] = {1432997174477.0 / 9575080441755.0, 5161836677717.0 / 13612068292357.0,
                       1720146321549.0 / 2090206949498.0, 3134564353537.0 / 4481467310338.0,
                       2277821191437.0 / 14882151754819.0};
const double RKC[5] = {0.0, 1432997174477.0 / 9575080441755.0, 2526269341429.0 / 6820363962896.0,
                       2006345519317.0 / 3224310063776.0, 2802321613138.0 / 2924317926251.0};


// ---------------------------------------------------------------- O12: exponential element filter (eq. 52)
// 1-D nodal filter matrix F = V diag(sigma) V^-1, V_ij = P_j(xi_i) (Legendre modes at the LGL nodes),
// sigma_j = exp(-alpha (j / N)^s): eta = mode number / polynomial order (R26), s = filter order, alpha = -log(eps_M).
void filter_matrix(int N, const double* xi, int order, double alpha, double (*F)[MAXNQ]) {
  const int Nq = N + 1;
  double V[MAXNQ][MAXNQ], Vi[MAXNQ][MAXNQ];
  for (int i = 0; i < Nq; ++i)
    for (int j = 0; j < Nq; ++j) { double P, dP; legendre(j, xi[i], P, dP); V[i][j] = P; }
  // inverse by Gauss-Jordan with partial pivoting
  double A[MAXNQ][2 * MAXNQ];
  for (int i = 0; i < Nq; ++i)
    for (int j = 0; j < Nq; ++j) { A[i][j] = V[i][j]; A[i][Nq + j] = (i == j) ? 1.0 : 0.0; }
  for (int col = 0; col < Nq; ++col) {
    int piv = col;
    for (int r = col + 1; r < Nq; ++r) if (std::fabs(A[r][col]) > std::fabs(A[piv][col])) piv = r;
    for (int j = 0; j < 2 * Nq; ++j) std::swap(A[col][j], A[piv][j]);
    double d = A[col][col];
    for (int j = 0; j < 2 * Nq; ++j) A[col][j] /= d;
    for (int r = 0; r < Nq; ++r)
      if (r != col) { double f = A[r][col]; for (int j = 0; j < 2 * Nq; ++j) A[r][j] -= f * A[col][j]; }
  }
  for (int i = 0; i < Nq; ++i) for (int j = 0; j < Nq; ++j) Vi[i][j] = A[i][Nq + j];
  for (int i = 0; i < Nq; ++i)
    for (int j = 0; j < Nq; ++j) {
      double a = 0;
      for (int m = 0; m < Nq; ++m) a += V[i][m] * std::exp(-alpha * std::pow((double)m / N, order)) * Vi[m][j];
      F[i][j] = a;
    }
}

// Q <- Q_ref + (F x F x F)(Q - Q_ref) on every element and prognostic field: "applied to perturbations of the prognostic
// variables from the balanced background state"; Q_ref = (rho_r, 0, rhoe_r, rhoq_r), zero without reference.
void apply_filter(const Ctx& c, double* Q) {
  const int Nq = c.Nq, Np = c.Np, nv = c.nvar;
#pragma omp parallel for schedule(static)
  for (int64_t e = 0; e < c.Ne; ++e) {
    std::vector<double> a(Np), b(Np), ref(Np);
    for (int v = 0; v < nv; ++v) {
      for (int n = 0; n < Np; ++n) {
        size_t id = (size_t)e * Np + n;
        ref[n] = 0.0;
        if (c.use_ref) ref[n] = (v == 0) ? c.ref_rho[id] : (v == 4) ? c.ref_rhoe[id] : (v == 5) ? c.ref_rhoq[id] : 0.0;
        a[n] = Q[id * nv + v] - ref[n];
      }
      for (int k = 0; k < Nq; ++k) for (int j = 0; j < Nq; ++j) for (int i = 0; i < Nq; ++i) {
        double t = 0; for (int m = 0; m < Nq; ++m) t += c.Filt[i][m] * a[m + Nq * (j + Nq * k)];
        b[i + Nq * (j + Nq * k)] = t;
      }
      for (int k = 0; k < Nq; ++k) for (int j = 0; j < Nq; ++j) for (int i = 0; i < Nq; ++i) {
        double t = 0; for (int m = 0; m < Nq; ++m) t += c.Filt[j][m] * b[i + Nq * (m + Nq * k)];
        a[i + Nq * (j + Nq * k)] = t;
      }
      for (int k = 0; k < Nq; ++k) for (int j = 0; j < Nq; ++j) for (int i = 0; i < Nq; ++i) {
        double t = 0; for (int m = 0; m < Nq; ++m) t += c.Filt[k][m] * a[i + Nq * (j + Nq * m)];
        b[i + Nq * (j + Nq * k)] = t;
      }
      for (int n = 0; n < Np; ++n) Q[((size_t)e * Np + n) * nv + v] = ref[n] + b[n];
    }
  }
}

// ---------------------------------------------------------------- O9/O13: 2N-storage Runge-Kutta with any coefficient table
// for s: dU <- A_s dU + dt RHS(U); U <- U + B_s dU; the element filter, when enabled, follows every step.
void lsrk_steps(const Ctx& c, double* Q, double dt, int nsteps, int nstages, const double* A, const double* B) {
  size_t n = (size_t)c.Ne * c.Np * c.nvar;
  std::vector<double> dU(n, 0.0), R(n);
  for (int step = 0; step < nsteps; ++step) {
    for (int s = 0; s < nstages; ++s) {
      rhs_all(c, Q, R.data(), 0);
      for (size_t i = 0; i < n; ++i) { dU[i] = A[s] * dU[i] + dt * R[i]; Q[i] = Q[i] + B[s] * dU[i]; }
    }
    if (c.filter_order > 0) apply_filter(c, Q);
  }
}

}  // namespace

// ---------------------------------------------------------------- O14: density-weighted horizontal statistics (App. B)
// Levels: every nodal zeta-plane of every element layer, l = ez * Nq + k (the planes of an element interface appear twice,
// once from each side: the DG solution is double-valued there).  <a>_l = sum W a / sum W over the nodes of the plane, with
// the area element of the zeta = const surface as weight, W = w_i w_j |Ja^3| ("metric terms accounted for").
// phi = u, v, w, h_tot, q_t, theta_v.  out[l][20] = <z>, <rho>, phibar (B1) x6, (w'phi')bar (B2) x6, (phi'^2)bar (B4) x6
// with phi' = phi - phibar (B3), w' = w - wbar.
constexpr int NPROF = 20;
void favre_profiles(const Ctx& c, const double* Q, double* out) {
  const int Nq = c.Nq, nlev = c.ne[2] * Nq;
  std::vector<double> sumW(nlev, 0.0);
  for (int l = 0; l < nlev * NPROF; ++l) out[l] = 0.0;
  // pass 1: <z>, <rho>, <rho phi>
  for (int pass = 0; pass < 2; ++pass) {
    for (int ez = 0; ez < c.ne[2]; ++ez)
      for (int ey = 0; ey < c.ne[1]; ++ey)
        for (int ex = 0; ex < c.ne[0]; ++ex) {
          int64_t e = elem_index(c, ex, ey, ez);
          Geo g; elem_geo(c, e, g);
          for (int n = 0; n < c.Np; ++n) {
            int i = n % Nq, j = (n / Nq) % Nq, k = n / (Nq * Nq);
            int l = ez * Nq + k;
            const double* a3 = g.Ja + 9 * n + 6;
            double W = c.w[i] * c.w[j] * std::sqrt(a3[0] * a3[0] + a3[1] * a3[1] + a3[2] * a3[2]);
            Prim P = prim_at(c, Q, e, n, g.x[3 * n + 2]);
            double phi[6]; grad_vars(P, phi);
            double* o = out + (size_t)l * NPROF;
            if (pass == 0) {
              sumW[l] += W;
              o[0] += W * g.x[3 * n + 2];
              o[1] += W * P.rho;
              for (int m = 0; m < 6; ++m) o[2 + m] += W * P.rho * phi[m];
            } else {
              double wp = phi[2] - o[2 + 2];
              for (int m = 0; m < 6; ++m) {
                double fp = phi[m] - o[2 + m];
                o[8 + m] += W * P.rho * wp * fp;
                o[14 + m] += W * P.rho * fp * fp;
              }
            }
          }
        }
    for (int l = 0; l < nlev; ++l) {
      double* o = out + (size_t)l * NPROF;
      if (pass == 0) {
        o[0] /= sumW[l]; o[1] /= sumW[l];                                  // <z>, <rho>
        for (int m = 0; m < 6; ++m) o[2 + m] = (o[2 + m] / sumW[l]) / o[1];   // (B1)
      } else {
        for (int m = 0; m < 12; ++m) o[8 + m] = (o[8 + m] / sumW[l]) / o[1];  // (B2), (B4)
      }
    }
  }
}

// ================================================================= C ABI (ctypes)
extern "C" {

struct odg_params {
  int32_t N;
  int32_t ne[3];
  double lo[3], hi[3];
  int32_t bc[3];
  int32_t nvar;
  int32_t geom;
  const double* zsfc_nodes;
  const double* xyz;
  double R_d, c_vd, R_v, c_vv, T_0, I_v0, grav;
  int32_t sgs;
  double C_s, Pr_t;
  int32_t use_ref;
  const double *ref_rho, *ref_rhoe, *ref_rhoq;
  double shf_bottom;
  int32_t cache_geometry;
  int32_t richardson;
  double p_0;
  double sponge_alpha, sponge_zs; int32_t sponge_gamma; double u_relax[3];
  int32_t filter_order; double filter_alpha;
  int32_t riemann;
  int32_t metric_form;
  double drag_cd, lhf_bottom, evap_bottom;
  int32_t satadj; double c_vl, p_tr, T_tr;
};

void odg_lgl(int N, double* xi, double* w) { lgl_nodes_weights(N, xi, w); }

void odg_dmat(int N, double* Dout /* [Nq][Nq] row-major */) {
  double xi[MAXNQ], w[MAXNQ], D[MAXNQ][MAXNQ];
  lgl_nodes_weights(N, xi, w); deriv_matrix(N, xi, D);
  for (int i = 0; i <= N; ++i) for (int j = 0; j <= N; ++j) Dout[i * (N + 1) + j] = D[i][j];
}

void odg_lsrk54_coeffs(double* A, double* B, double* C) {
  for (int s = 0; s < 5; ++s) { A[s] = RKA[s]; B[s] = RKB[s]; C[s] = RKC[s]; }
}

void* odg_create(const odg_params* p) {
  if (!p || p->N < 1 || p->N + 1 > MAXNQ - 1) return nullptr;
  Ctx* c = new Ctx();
  c->N = p->N; c->Nq = p->N + 1; c->Np = c->Nq * c->Nq * c->Nq;
  for (int d = 0; d < 3; ++d) { c->ne[d] = p->ne[d]; c->lo[d] = p->lo[d]; c->hi[d] = p->hi[d]; c->bc[d] = p->bc[d]; }
  c->Ne = (int64_t)c->ne[0] * c->ne[1] * c->ne[2];
  c->nvar = p->nvar; c->geom = p->geom;
  c->R_d = p->R_d; c->c_vd = p->c_vd; c->R_v = p->R_v; c->c_vv = p->c_vv; c->T_0 = p->T_0; c->I_v0 = p->I_v0;
  c->grav = p->grav; c->sgs = p->sgs; c->C_s = p->C_s; c->Pr_t = p->Pr_t; c->use_ref = p->use_ref;
  c->shf_bottom = p->shf_bottom;
  c->richardson = p->richardson; c->p_0 = p->p_0;
  c->sponge_alpha = p->sponge_alpha; c->sponge_zs = p->sponge_zs; c->sponge_gamma = p->sponge_gamma;
  for (int d = 0; d < 3; ++d) c->u_relax[d] = p->u_relax[d];
  c->filter_order = p->filter_order; c->filter_alpha = p->filter_alpha;
  c->riemann = p->riemann; c->metric_form = p->metric_form;
  c->drag_cd = p->drag_cd; c->lhf_bottom = p->lhf_bottom; c->evap_bottom = p->evap_bottom;
  c->satadj = p->satadj;
  if (p->c_vl > 0.0) c->c_vl = p->c_vl;
  if (p->p_tr > 0.0) c->p_tr = p->p_tr;
  if (p->T_tr > 0.0) c->T_tr = p->T_tr;
  lgl_nodes_weights(c->N, c->xi, c->w);
  deriv_matrix(c->N, c->xi, c->D);
  if (c->filter_order > 0) filter_matrix(c->N, c->xi, c->filter_order, c->filter_alpha, c->Filt);
  size_t nn = (size_t)c->Ne * c->Np;
  if (c->geom == 1) c->zsfc.assign(p->zsfc_nodes, p->zsfc_nodes + (size_t)c->ne[0] * c->Nq * c->ne[1] * c->Nq);
  if (c->geom == 2) c->xyz_in.assign(p->xyz, p->xyz + 3 * nn);
  if (c->use_ref) {
    c->ref_rho.assign(p->ref_rho, p->ref_rho + nn);
    c->ref_rhoe.assign(p->ref_rhoe, p->ref_rhoe + nn);
    if (c->nvar == 6) c->ref_rhoq.assign(p->ref_rhoq, p->ref_rhoq + nn);
  }
  if (p->cache_geometry) {
    c->cx.resize(nn * 3); c->cJa.resize(nn * 9); c->cJ.resize(nn); c->cDx.resize(nn * 3);
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < c->Ne; ++e)
      elem_geo_compute(*c, e, &c->cx[(size_t)e * c->Np * 3], &c->cJa[(size_t)e * c->Np * 9], &c->cJ[(size_t)e * c->Np],
                       &c->cDx[(size_t)e * c->Np * 3]);
    c->cached = true;
  }
  return c;
}

void odg_destroy(void* h) { delete (Ctx*)h; }

// coordinates xyz[e][n][3]
void odg_coords(void* h, double* xyz) {
  const Ctx& c = *(Ctx*)h;
#pragma omp parallel for schedule(static)
  for (int64_t e = 0; e < c.Ne; ++e) elem_nodes(c, e, xyz + (size_t)e * c.Np * 3);
}

// geometry of one element: Ja[n][d][cc], J[n], mass M[n] = w_i w_j w_k J, and per face-node
// sJn[f][b][a][3] = sJ * n (outward), lift[f][b][a] = sJ / (w_0 J)
void odg_elem_geometry(void* h, int64_t e, double* Ja, double* J, double* M, double* sJn, double* lift) {
  const Ctx& c = *(Ctx*)h;
  Geo g; elem_geo(c, e, g);
  const int Nq = c.Nq;
  for (int n = 0; n < c.Np; ++n) {
    for (int m = 0; m < 9; ++m) Ja[9 * n + m] = g.Ja[9 * n + m];
    J[n] = g.J[n];
    int i = n % Nq, j = (n / Nq) % Nq, k = n / (Nq * Nq);
    M[n] = c.w[i] * c.w[j] * c.w[k] * g.J[n];
  }
  for (int f = 0; f < 6; ++f)
    for (int b = 0; b < Nq; ++b)
      for (int a = 0; a < Nq; ++a) {
        int n = face_node(Nq, f, a, b, false);
        int d = f / 2; double sgn = (f % 2) ? 1.0 : -1.0;
        const double* A = g.Ja + 9 * n + 3 * d;
        double sJ = std::sqrt(A[0] * A[0] + A[1] * A[1] + A[2] * A[2]);
        for (int cc = 0; cc < 3; ++cc) sJn[((f * Nq + b) * Nq + a) * 3 + cc] = sgn * A[cc];
        lift[(f * Nq + b) * Nq + a] = sJ / (c.w[0] * g.J[n]);
      }
}

int64_t odg_neighbour(void* h, int64_t e, int f) { return neighbour(*(Ctx*)h, e, f); }

// diagonal of dx/dxi at the nodes of element e: dxd[n][3]
void odg_elem_dxd(void* h, int64_t e, double* dxd) {
  const Ctx& c = *(Ctx*)h;
  Geo g; elem_geo(c, e, g);
  for (int n = 0; n < 3 * c.Np; ++n) dxd[n] = g.dxd[n];
}

// pointwise thermodynamics: out = rho,u,v,w,q,T,p,pp,htot,c,theta_v,q_l
void odg_primitives(void* h, const double* Y, double z, int has_ref, double rr, double rer, double rqr, double* out) {
  const Ctx& c = *(Ctx*)h;
  Prim P = primitives(c, Y, z, has_ref != 0, rr, rer, rqr);
  out[0] = P.rho; out[1] = P.u[0]; out[2] = P.u[1]; out[3] = P.u[2]; out[4] = P.q; out[5] = P.T; out[6] = P.p;
  out[7] = P.pp; out[8] = P.htot; out[9] = P.c; out[10] = P.theta_v; out[11] = P.ql;
}
// saturation vapour pressure over liquid [Pa] (O15)
double odg_sat_vapor_pressure(void* h, double T) { return sat_vapor_pressure(*(Ctx*)h, T); }

// pointwise Rusanov flux n.F1* of two states at height z without reference state (pins: consistency, symmetry)
void odg_rusanov(void* h, const double* Ym, const double* Yp, const double* nrm, double z, double* Fstar) {
  const Ctx& c = *(Ctx*)h;
  Prim Pm = primitives(c, Ym, z, false, 0, 0, 0), Pp = primitives(c, Yp, z, false, 0, 0, 0);
  double F1m[6][3], F1p[6][3];
  flux_first_order(c, Ym, Pm, F1m); flux_first_order(c, Yp, Pp, F1p);
  numerical_flux(c, Ym, Pm, F1m, Yp, Pp, F1p, nrm, Fstar);   // Rusanov or HLLC, as the ctx says
}

// physical first-order flux F1[v][3] at a point (no reference state)
void odg_flux1(void* h, const double* Y, double z, double* F) {
  const Ctx& c = *(Ctx*)h;
  Prim P = primitives(c, Y, z, false, 0, 0, 0);
  double F1[6][3]; flux_first_order(c, Y, P, F1);
  for (int v = 0; v < c.nvar; ++v) for (int cc = 0; cc < 3; ++cc) F[v * 3 + cc] = F1[v][cc];
}

// second-order flux F2[v][3] at a point given the gradient G[6][3] (u, v, w, h_tot, q, theta_v), the metric
// determinant J and the diagonal dxd[3] of dx/dxi (mixing lengths of the Vreman model)
void odg_flux2(void* h, const double* Y, double z, const double* G, double J, const double* dxd, double* F, double* nu_t) {
  const Ctx& c = *(Ctx*)h;
  Prim P = primitives(c, Y, z, false, 0, 0, 0);
  double F2[6][3]; flux_second_order(c, Y, P, G, J, dxd, F2);
  for (int v = 0; v < c.nvar; ++v) for (int cc = 0; cc < 3; ++cc) F[v * 3 + cc] = F2[v][cc];
  *nu_t = eddy_viscosity(c, G, J, dxd, P.theta_v);
}

// BR1 gradient of the whole mesh: G[e][n][5][3]
void odg_gradient(void* h, const double* Q, double* G) {
  const Ctx& c = *(Ctx*)h;
  std::vector<double> G6((size_t)c.Ne * c.Np * NG3);
  gradient_all(c, Q, G6.data());
  for (size_t i = 0; i < (size_t)c.Ne * c.Np; ++i)
    for (int m = 0; m < 15; ++m) G[i * 15 + m] = G6[i * NG3 + m];
}
// the same with the sixth gradient variable theta_v: G[e][n][6][3]
void odg_gradient6(void* h, const double* Q, double* G) { gradient_all(*(Ctx*)h, Q, G); }

// dQ[e][n][v] = RHS(Q); form 0 = weak (eq. 26), 1 = strong (eq. 32)
void odg_rhs(void* h, const double* Q, double* dQ, int form) { rhs_all(*(Ctx*)h, Q, dQ, form); }

// RHS of selected elements only (full-size sampled parity): out[s][n][v] for elems[s]
void odg_rhs_elements(void* h, const double* Q, const int64_t* elems, int64_t nel, double* out) {
  const Ctx& c = *(Ctx*)h;
#pragma omp parallel for schedule(dynamic)
  for (int64_t s = 0; s < nel; ++s) {
    int64_t e = elems[s];
    std::vector<double> Ge, Gnb[6];
    const double* Gn[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    if (c.sgs) {
      Ge.resize((size_t)c.Np * NG3); gradient_element(c, Q, e, Ge.data());
      for (int f = 0; f < 6; ++f) {
        int64_t en = neighbour(c, e, f);
        if (en >= 0) { Gnb[f].resize((size_t)c.Np * NG3); gradient_element(c, Q, en, Gnb[f].data()); Gn[f] = Gnb[f].data(); }
      }
    }
    rhs_element(c, Q, e, c.sgs ? Ge.data() : nullptr, Gn, 0, out + (size_t)s * c.Np * c.nvar);
  }
}

// LSRK54: for s: dU <- A_s dU + dt RHS(U, t + C_s dt); U <- U + B_s dU
void odg_lsrk54(void* h, double* Q, double t, double dt, int nsteps) {
  (void)t;
  lsrk_steps(*(Ctx*)h, Q, dt, nsteps, 5, RKA, RKB);
}

// the same for any 2N-storage coefficient table (A_1 must be 0), e.g. the 14-stage scheme the paper ran
void odg_lsrk_table(void* h, double* Q, double dt, int nsteps, int nstages, const double* A, const double* B) {
  lsrk_steps(*(Ctx*)h, Q, dt, nsteps, nstages, A, B);
}

// exponential element filter (eq. 52) applied once, in place; the 1-D filter matrix [Nq][Nq] row-major
void odg_filter(void* h, double* Q) { apply_filter(*(Ctx*)h, Q); }
void odg_filter_matrix(int N, int order, double alpha, double* Fout) {
  double xi[MAXNQ], w[MAXNQ], F[MAXNQ][MAXNQ];
  lgl_nodes_weights(N, xi, w); filter_matrix(N, xi, order, alpha, F);
  for (int i = 0; i <= N; ++i) for (int j = 0; j <= N; ++j) Fout[i * (N + 1) + j] = F[i][j];
}

// forward Euler: U <- U + dt RHS(U)
void odg_euler(void* h, double* Q, double dt, int nsteps) {
  const Ctx& c = *(Ctx*)h;
  size_t n = (size_t)c.Ne * c.Np * c.nvar;
  std::vector<double> R(n);
  for (int step = 0; step < nsteps; ++step) {
    rhs_all(c, Q, R.data(), 0);
    for (size_t i = 0; i < n; ++i) Q[i] += dt * R[i];
  }
}

// one LSRK stage on given residual storage (used for timing the oracle: gradient + RHS + update)
void odg_lsrk54_stage(void* h, double* Q, double* dU, double dt, int s) {
  const Ctx& c = *(Ctx*)h;
  size_t n = (size_t)c.Ne * c.Np * c.nvar;
  std::vector<double> R(n);
  rhs_all(c, Q, R.data(), 0);
  for (size_t i = 0; i < n; ++i) { dU[i] = RKA[s] * dU[i] + dt * R[i]; Q[i] = Q[i] + RKB[s] * dU[i]; }
}

// diagnostics (eq. 57, 61, 62): out = mass, energy, water, kinetic (volume mean of |u|^2/2), max(|u|+c),
// min node spacing, volume, count of non-finite state values
void odg_diagnostics(void* h, const double* Q, double* out) {
  const Ctx& c = *(Ctx*)h;
  const int Nq = c.Nq;
  double mass = 0, energy = 0, water = 0, ke = 0, vol = 0, wmax = 0, dxmin = 1e300, nonf = 0;
  for (int64_t e = 0; e < c.Ne; ++e) {
    Geo g; elem_geo(c, e, g);
    for (int n = 0; n < c.Np; ++n) {
      int i = n % Nq, j = (n / Nq) % Nq, k = n / (Nq * Nq);
      double M = c.w[i] * c.w[j] * c.w[k] * g.J[n];
      const double* Y = Q + ((size_t)e * c.Np + n) * c.nvar;
      for (int v = 0; v < c.nvar; ++v) if (!std::isfinite(Y[v])) nonf += 1;
      Prim P = prim_at(c, Q, e, n, g.x[3 * n + 2]);
      mass += M * Y[0]; energy += M * Y[4]; if (c.nvar == 6) water += M * Y[5];
      ke += M * 0.5 * (P.u[0] * P.u[0] + P.u[1] * P.u[1] + P.u[2] * P.u[2]);
      vol += M;
      double sp = std::sqrt(P.u[0] * P.u[0] + P.u[1] * P.u[1] + P.u[2] * P.u[2]) + P.c;
      if (sp > wmax) wmax = sp;
      // distance to the next node in each direction
      int nb[3] = {(i + 1 < Nq) ? n + 1 : -1, (j + 1 < Nq) ? n + Nq : -1, (k + 1 < Nq) ? n + Nq * Nq : -1};
      for (int d = 0; d < 3; ++d)
        if (nb[d] >= 0) {
          double dx = 0;
          for (int cc = 0; cc < 3; ++cc) { double t = g.x[3 * nb[d] + cc] - g.x[3 * n + cc]; dx += t * t; }
          dx = std::sqrt(dx);
          if (dx < dxmin) dxmin = dx;
        }
    }
  }
  out[0] = mass; out[1] = energy; out[2] = water; out[3] = ke / vol; out[4] = wmax; out[5] = dxmin; out[6] = vol; out[7] = nonf;
}

// density-weighted horizontal statistics (App. B): out[Ez*Nq][20], see favre_profiles
void odg_profiles(void* h, const double* Q, double* out) { favre_profiles(*(Ctx*)h, Q, out); }

int odg_num_threads() {
  int n = 1;
#ifdef _OPENMP
#pragma omp parallel
  {
#pragma omp single
    n = omp_get_num_threads();
  }
#endif
  return n;
}

}  // extern "C"
