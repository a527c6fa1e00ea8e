// cm_dg_lib.cu -- host side of the C ABI in include/cm_dg.h plus the setup / diagnostics kernels:
//   a0  LGL nodes, weights, derivative matrix; element ordering and connectivity; metric terms
//       (eq. 24) by a CUDA kernel; reference-state tables
//   a6  conservation integrals (eq. 57, 61, 62)
// The hot kernels live in cm_dg_kernels.cuh.  There is no CPU fallback anywhere in this file: every
// entry point that computes needs a CUDA device and fails with CM_DG_ECUDA without one.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/cm_dg.h"
#include "cm_dg_internal.h"
#include "cm_dg_physics.cuh"

namespace {

thread_local std::string g_err = "";
int fail(int code, const std::string& msg) { g_err = msg; return code; }
#define CM_CUDA(call)                                                                                    \
  do {                                                                                                   \
    cudaError_t err__ = (call);                                                                          \
    if (err__ != cudaSuccess)                                                                            \
      return fail(err__ == cudaErrorMemoryAllocation ? CM_DG_ENOMEM : CM_DG_ECUDA,                       \
                  std::string(#call) + ": " + cudaGetErrorString(err__));                                \
  } while (0)

// LSRK54 of Carpenter & Kennedy (1994), 2N-storage (5,4) scheme (P:L286 cites the family).
const double kRKA[5] = {0.0, -567301805773.0 / 1357537059087.0, -2404267990393.0 / 2016746695238.0,
                        -3550918686646.0 / 2091501179385.0, -1275806237668.0 / 842570457699.0};
const double kRKB[5] = {1432997174477.0 / 9575080441755.0, 5161836677717.0 / 13612068292357.0,
                        1720146321549.0 / 2090206949498.0, 3134564353537.0 / 4481467310338.0,
                        2277821191437.0 / 14882151754819.0};

// ------------------------------------------------------------------ a0: 1-D operators
// LGL points as the roots of q(x) = P_{N+1}(x) - P_{N-1}(x) (proportional to (1 - x^2) P_N'(x)), Newton in
// long double; weights 2 / (N (N+1) P_N^2); D from barycentric weights with the negative-sum diagonal.
void lgl_operators(int N, double* xi, double* w, double (*D)[CM_MAXNQ]) {
  const int Nq = N + 1;
  std::vector<long double> x(Nq);
  const long double pi = 3.14159265358979323846264338327950288L;
  auto legendre3 = [&](long double t, long double& Pm1, long double& P0, long double& Pp1) {
    long double a = 1.0L, b = t;   // P_0, P_1
    for (int n = 1; n < N; ++n) { long double c = ((2 * n + 1) * t * b - n * a) / (n + 1); a = b; b = c; }
    // now a = P_{N-1}, b = P_N
    Pm1 = a; P0 = b; Pp1 = ((2 * N + 1) * t * b - N * a) / (N + 1);
  };
  for (int i = 0; i < Nq; ++i) {
    long double t = -std::cos(pi * i / N);
    if (i == 0) t = -1.0L; else if (i == N) t = 1.0L;
    else
      for (int it = 0; it < 60; ++it) {
        long double a, b, c; legendre3(t, a, b, c);
        long double q = c - a, dq = (2 * N + 1) * b;          // q' = (2N+1) P_N
        long double dt = q / dq; t -= dt;
        if (fabsl(dt) < 1e-20L) break;
      }
    x[i] = t;
  }
  for (int i = 0; i < Nq / 2; ++i) { long double m = 0.5L * (x[N - i] - x[i]); x[i] = -m; x[N - i] = m; }
  if (N % 2 == 0) x[N / 2] = 0.0L;
  std::vector<long double> bw(Nq);
  for (int i = 0; i < Nq; ++i) {
    long double a, b, c; legendre3(x[i], a, b, c);
    xi[i] = (double)x[i];
    w[i] = (double)(2.0L / (N * (N + 1.0L) * b * b));
    long double prod = 1.0L;
    for (int l = 0; l < Nq; ++l) if (l != i) prod *= (x[i] - x[l]);
    bw[i] = 1.0L / prod;
  }
  for (int i = 0; i < Nq; ++i) {
    long double s = 0.0L;
    for (int j = 0; j < Nq; ++j) {
      if (i == j) continue;
      long double dij = (bw[j] / bw[i]) / (x[i] - x[j]);
      D[i][j] = (double)dij; s += dij;
    }
    D[i][i] = (double)(-s);
  }
}

// 1-D nodal matrix of the exponential filter of eq. (52): F = V diag(sigma) V^-1 with V_ij = P_j(xi_i) (Legendre modes at
// the LGL nodes) and sigma_j = exp(-alpha (j / N)^s) (eta = mode number / polynomial order, reading R26); long double.
void filter_operator(int N, const double* xi, int order, double alpha, double (*F)[CM_MAXNQ]) {
  const int Nq = N + 1;
  long double A[CM_MAXNQ][2 * CM_MAXNQ], V[CM_MAXNQ][CM_MAXNQ];
  for (int i = 0; i < Nq; ++i) {
    long double a = 1.0L, b = xi[i];
    for (int j = 0; j < Nq; ++j) {
      V[i][j] = (j == 0) ? a : b;
      if (j >= 1) { long double cnx = ((2 * j + 1) * (long double)xi[i] * b - j * a) / (j + 1); a = b; b = cnx; }
    }
  }
  for (int i = 0; i < Nq; ++i)
    for (int j = 0; j < Nq; ++j) { A[i][j] = V[i][j]; A[i][Nq + j] = (i == j) ? 1.0L : 0.0L; }
  for (int col = 0; col < Nq; ++col) {
    int piv = col;
    for (int r = col + 1; r < Nq; ++r) if (fabsl(A[r][col]) > fabsl(A[piv][col])) piv = r;
    for (int j = 0; j < 2 * Nq; ++j) std::swap(A[col][j], A[piv][j]);
    const long double d = A[col][col];
    for (int j = 0; j < 2 * Nq; ++j) A[col][j] /= d;
    for (int r = 0; r < Nq; ++r)
      if (r != col) { const long double f = A[r][col]; for (int j = 0; j < 2 * Nq; ++j) A[r][j] -= f * A[col][j]; }
  }
  for (int i = 0; i < Nq; ++i)
    for (int j = 0; j < Nq; ++j) {
      long double acc = 0.0L;
      for (int m = 0; m < Nq; ++m) acc += V[i][m] * expl(-(long double)alpha * powl((long double)m / N, order)) * A[m][Nq + j];
      F[i][j] = (double)acc;
    }
}

// ------------------------------------------------------------------ small kernels
struct GeoArgs {
  int Nq, Np, geom;
  long long Ne, stride;
  int ne[3];
  double lo[3], hi[3], h[3];
  const int* lex;         // [Ne] lexicographic id of library element
  const double* zsfc;     // geom 1
  const double* xyz_user; // geom 2: [3][stride] library order
  double xi[CM_MAXNQ], w[CM_MAXNQ], D[CM_MAXNQ][CM_MAXNQ];
  double cs, grav;
  int N, metric_form;          // polynomial order; 0 cross-product | 1 curl-invariant metric terms
  double sp_alpha, sp_zs; int sp_gamma;   // Rayleigh sponge (A5)
};

__device__ inline void node_xyz(const GeoArgs& a, long long e, int n, double* X) {
  if (a.geom == 2) {
    for (int d = 0; d < 3; ++d) X[d] = a.xyz_user[d * a.stride + e * a.Np + n];
    return;
  }
  const int lex = a.lex[e];
  const int ec[3] = {lex % a.ne[0], (lex / a.ne[0]) % a.ne[1], lex / (a.ne[0] * a.ne[1])};
  const int ijk[3] = {n % a.Nq, (n / a.Nq) % a.Nq, n / (a.Nq * a.Nq)};
  for (int d = 0; d < 3; ++d) X[d] = a.lo[d] + (ec[d] + 0.5 * (a.xi[ijk[d]] + 1.0)) * a.h[d];
  if (a.geom == 1) {
    const double zs = a.zsfc[(long long)(ec[1] * a.Nq + ijk[1]) * (a.ne[0] * a.Nq) + ec[0] * a.Nq + ijk[0]];
    X[2] += zs * (a.hi[2] - X[2]) / (a.hi[2] - a.lo[2]);      // linear decay to a flat lid
  }
}

__global__ void coords_kernel(const __grid_constant__ GeoArgs a, double* __restrict__ xyz) {
  const long long e = blockIdx.x;
  for (int n = threadIdx.x; n < a.Np; n += blockDim.x) {
    double X[3]; node_xyz(a, e, n, X);
    for (int d = 0; d < 3; ++d) xyz[d * a.stride + e * a.Np + n] = X[d];
  }
}

// metric terms of one element per block: geo = Ja[9], 1/J, z, (C_s Delta)^2; chk[e] = {min J, metric-identity
// residual / max|Ja|, min node spacing}
__device__ inline double sponge_tau(double alpha, double zs, int gamma, double ztop, double z) {
  // tau_s = alpha sin^gamma(pi/2 (z - z_s) / (z_top - z_s)) for z > z_s   (A5 with reading R18)
  if (!(alpha > 0.0) || !(z > zs)) return 0.0;
  return alpha * pow(sin(0.5 * 3.14159265358979323846 * (z - zs) / (ztop - zs)), (double)gamma);
}

__global__ void metrics_kernel(const __grid_constant__ GeoArgs a, double* __restrict__ geo, double* __restrict__ chk) {
  extern __shared__ double sh[];
  double* X = sh;                 // [3][Np]
  double* JA = sh + 3 * a.Np;     // [9][Np]
  double* DX = JA + 9 * a.Np;     // [9][Np]  d x_c / d xi_d at [3 d + c]  (curl form)
  double* V = DX + 9 * a.Np;      // [3][Np]  X_l d X_m / d xi_d           (curl form)
  double* red = V + 3 * a.Np;     // [4][blockDim]
  const long long e = blockIdx.x;
  const int Nq = a.Nq, Np = a.Np;
  for (int n = threadIdx.x; n < Np; n += blockDim.x) {
    double P[3]; node_xyz(a, e, n, P);
    for (int d = 0; d < 3; ++d) X[d * Np + n] = P[d];
  }
  __syncthreads();
  double minJ = 1e300, mindx = 1e300, amax = 0.0;
  for (int n = threadIdx.x; n < Np; n += blockDim.x) {
    const int i = n % Nq, j = (n / Nq) % Nq, k = n / (Nq * Nq);
    double xr[3] = {0, 0, 0}, xs[3] = {0, 0, 0}, xt[3] = {0, 0, 0};
    // coordinates relative to the element's first node: same derivative, no rounding of the offset from the origin
    for (int m = 0; m < Nq; ++m)
      for (int d = 0; d < 3; ++d) {
        xr[d] += a.D[i][m] * (X[d * Np + m + Nq * (j + Nq * k)] - X[d * Np]);
        xs[d] += a.D[j][m] * (X[d * Np + i + Nq * (m + Nq * k)] - X[d * Np]);
        xt[d] += a.D[k][m] * (X[d * Np + i + Nq * (j + Nq * m)] - X[d * Np]);
      }
    for (int d = 0; d < 3; ++d) { DX[d * Np + n] = xr[d]; DX[(3 + d) * Np + n] = xs[d]; DX[(6 + d) * Np + n] = xt[d]; }
    double A[9];
    A[0] = xs[1] * xt[2] - xs[2] * xt[1]; A[1] = xs[2] * xt[0] - xs[0] * xt[2]; A[2] = xs[0] * xt[1] - xs[1] * xt[0];
    A[3] = xt[1] * xr[2] - xt[2] * xr[1]; A[4] = xt[2] * xr[0] - xt[0] * xr[2]; A[5] = xt[0] * xr[1] - xt[1] * xr[0];
    A[6] = xr[1] * xs[2] - xr[2] * xs[1]; A[7] = xr[2] * xs[0] - xr[0] * xs[2]; A[8] = xr[0] * xs[1] - xr[1] * xs[0];
    const double J = xr[0] * A[0] + xr[1] * A[1] + xr[2] * A[2];
    const long long idx = e * Np + n;
    for (int m = 0; m < 9; ++m) JA[m * Np + n] = A[m];
    geo[9 * a.stride + idx] = 1.0 / J;
    geo[10 * a.stride + idx] = X[2 * Np + n];
    const double delta = cbrt(8.0 * J) / (Nq - 1);              // filter width, reading R7
    geo[11 * a.stride + idx] = (a.cs * delta) * (a.cs * delta);
    const double dm[3] = {2.0 * fabs(xr[0]) / a.N, 2.0 * fabs(xs[1]) / a.N, 2.0 * fabs(xt[2]) / a.N};   // mixing lengths (eq. 39c, R24)
    for (int m = 0; m < 3; ++m) geo[(12 + m) * a.stride + idx] = dm[m] * dm[m];
    geo[15 * a.stride + idx] = sponge_tau(a.sp_alpha, a.sp_zs, a.sp_gamma, a.hi[2], X[2 * Np + n]);
    minJ = fmin(minJ, J);
    const int nb[3] = {(i + 1 < Nq) ? n + 1 : -1, (j + 1 < Nq) ? n + Nq : -1, (k + 1 < Nq) ? n + Nq * Nq : -1};
    for (int d = 0; d < 3; ++d)
      if (nb[d] >= 0) {
        double s = 0;
        for (int c = 0; c < 3; ++c) { const double t = X[c * Np + nb[d]] - X[c * Np + n]; s += t * t; }
        mindx = fmin(mindx, sqrt(s));
      }
  }
  __syncthreads();
  if (a.metric_form == 1) {
    // curl-invariant form (Kopriva 2006): Ja^i_n = -xhat_i . curl_xi( I_N( X_l grad_xi X_m ) ), (n, m, l) cyclic: the
    // discrete metric identities then hold on fully 3-D warps
    for (int nn = 0; nn < 3; ++nn) {
      const int mm = (nn + 1) % 3, ll = (nn + 2) % 3;
      for (int n = threadIdx.x; n < Np; n += blockDim.x)
        for (int d = 0; d < 3; ++d) V[d * Np + n] = (X[ll * Np + n] - X[ll * Np]) * DX[(3 * d + mm) * Np + n];
      __syncthreads();
      for (int n = threadIdx.x; n < Np; n += blockDim.x) {
        const int i = n % Nq, j = (n / Nq) % Nq, k = n / (Nq * Nq);
        double dV[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};      // dV[a][d] = d V_d / d xi_a
        for (int m = 0; m < Nq; ++m)
          for (int d = 0; d < 3; ++d) {
            dV[0][d] += a.D[i][m] * V[d * Np + m + Nq * (j + Nq * k)];
            dV[1][d] += a.D[j][m] * V[d * Np + i + Nq * (m + Nq * k)];
            dV[2][d] += a.D[k][m] * V[d * Np + i + Nq * (j + Nq * m)];
          }
        JA[(0 + nn) * Np + n] = -(dV[1][2] - dV[2][1]);
        JA[(3 + nn) * Np + n] = -(dV[2][0] - dV[0][2]);
        JA[(6 + nn) * Np + n] = -(dV[0][1] - dV[1][0]);
      }
      __syncthreads();
    }
  }
  for (int n = threadIdx.x; n < Np; n += blockDim.x)
    for (int m = 0; m < 9; ++m) { const double v = JA[m * Np + n]; geo[m * a.stride + e * Np + n] = v; amax = fmax(amax, fabs(v)); }
  __syncthreads();
  double res = 0.0;
  for (int n = threadIdx.x; n < Np; n += blockDim.x) {
    const int i = n % Nq, j = (n / Nq) % Nq, k = n / (Nq * Nq);
    for (int c = 0; c < 3; ++c) {
      double r = 0.0;
      for (int m = 0; m < Nq; ++m)
        r += a.D[i][m] * JA[(0 + c) * Np + m + Nq * (j + Nq * k)] + a.D[j][m] * JA[(3 + c) * Np + i + Nq * (m + Nq * k)] +
             a.D[k][m] * JA[(6 + c) * Np + i + Nq * (j + Nq * m)];
      res = fmax(res, fabs(r));
    }
  }
  __syncthreads();
  red[threadIdx.x] = minJ; red[blockDim.x + threadIdx.x] = res; red[2 * blockDim.x + threadIdx.x] = mindx;
  double* red4 = red + 3 * blockDim.x; red4[threadIdx.x] = amax;
  __syncthreads();
  if (threadIdx.x == 0) {
    double mj = 1e300, rr = 0, md = 1e300, am = 0;
    for (int t = 0; t < blockDim.x; ++t) {
      mj = fmin(mj, red[t]); rr = fmax(rr, red[blockDim.x + t]); md = fmin(md, red[2 * blockDim.x + t]); am = fmax(am, red4[t]);
    }
    chk[3 * e] = mj; chk[3 * e + 1] = rr / fmax(am, 1e-300); chk[3 * e + 2] = md;
  }
}

__global__ void flat_metrics_fill(long long n, long long stride, const double cA0, const double cA1, const double cA2,
                                  const double J, double* __restrict__ Ja, double* __restrict__ Jout) {
  const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (t >= n) return;
  for (int m = 0; m < 9; ++m) Ja[m * stride + t] = 0.0;
  Ja[0 * stride + t] = cA0; Ja[4 * stride + t] = cA1; Ja[8 * stride + t] = cA2;
  Jout[t] = J;
}

__global__ void general_metrics_copy(long long n, long long stride, const double* __restrict__ geo,
                                     double* __restrict__ Ja, double* __restrict__ Jout) {
  const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (t >= n) return;
  for (int m = 0; m < 9; ++m) Ja[m * stride + t] = geo[m * stride + t];
  Jout[t] = 1.0 / geo[9 * stride + t];
}

// a6: per-block partial sums {mass, energy, water, M |u|^2 / 2, M, max(|u|+c), nonfinite}
struct DiagArgs {
  int Nq, Np, nvar, general, use_ref, satadj;
  long long Ne, stride;
  const double* Q; const double* geo; const int* erow; const double* ztab;
  double Jflat; double w[CM_MAXNQ];
  CmThermo th;
};

__global__ void diag_kernel(const __grid_constant__ DiagArgs a, double* __restrict__ part) {
  extern __shared__ double sh[];
  const long long e = blockIdx.x;
  double s[7] = {0, 0, 0, 0, 0, 0, 0};
  for (int n = threadIdx.x; n < a.Np; n += blockDim.x) {
    const int i = n % a.Nq, j = (n / a.Nq) % a.Nq, k = n / (a.Nq * a.Nq);
    const long long idx = e * a.Np + n;
    double Y[6] = {0, 0, 0, 0, 0, 0};
    for (int v = 0; v < a.nvar; ++v) { Y[v] = a.Q[v * a.stride + idx]; if (!isfinite(Y[v])) s[6] += 1.0; }
    const double J = a.general ? 1.0 / a.geo[9 * a.stride + idx] : a.Jflat;
    const double Phi = a.general ? a.th.grav * a.geo[10 * a.stride + idx] : a.ztab[(long long)(a.erow[e] + k) * CM_ZTAB_W];
    const double M = a.w[i] * a.w[j] * a.w[k] * J;
    const double ir = 1.0 / Y[0];
    const double u2 = (Y[1] * Y[1] + Y[2] * Y[2] + Y[3] * Y[3]) * ir * ir;
    const double q = (a.nvar == 6) ? Y[5] * ir : 0.0;
    double cvm = a.th.c_vd + a.th.b * q, Rm = a.th.R_d + a.th.a * q;
    const double eint = Y[4] * ir - 0.5 * u2 - Phi;
    double T = a.th.T_0 + (eint - q * a.th.I_v0) / cvm;
    if (a.satadj) T = cm_sat_pressure(a.th, Y[0], eint, q, Rm, cvm) / (Y[0] * Rm);
    const double c = sqrt((1.0 + Rm / cvm) * Rm * T);
    s[0] += M * Y[0]; s[1] += M * Y[4]; s[2] += M * Y[5]; s[3] += M * 0.5 * u2; s[4] += M;
    s[5] = fmax(s[5], sqrt(u2) + c);
  }
  for (int m = 0; m < 7; ++m) sh[m * blockDim.x + threadIdx.x] = s[m];
  __syncthreads();
  if (threadIdx.x == 0) {
    double r[7] = {0, 0, 0, 0, 0, 0, 0};
    for (int t = 0; t < blockDim.x; ++t)
      for (int m = 0; m < 7; ++m) r[m] = (m == 5) ? fmax(r[m], sh[m * blockDim.x + t]) : r[m] + sh[m * blockDim.x + t];
    for (int m = 0; m < 7; ++m) part[7 * e + m] = r[m];
  }
}

// eq. (52): Q <- Q_ref + (F x F x F)(Q - Q_ref), one element per block, one field at a time through shared memory
struct FilterArgs {
  int Nq, Np, nvar, general, use_ref;
  long long stride;
  double* Q; const int* erow; const double* ztab; const double* ref;
  double F[CM_MAXNQ][CM_MAXNQ];
};

__global__ void filter_kernel(const __grid_constant__ FilterArgs a) {
  extern __shared__ double sh[];
  double* u = sh; double* w = sh + a.Np;
  const long long e = blockIdx.x;
  const int Nq = a.Nq, Np = a.Np;
  for (int v = 0; v < a.nvar; ++v) {
    for (int n = threadIdx.x; n < Np; n += blockDim.x) {
      const long long idx = e * Np + n;
      double r = 0.0;
      if (a.use_ref && (v == 0 || v >= 4)) {
        const int col = (v == 0) ? 0 : (v == 4) ? 1 : 2;                   // rho_r, rhoe_r, rhoq_r
        r = a.general ? a.ref[col * a.stride + idx] : a.ztab[(long long)(a.erow[e] + n / (Nq * Nq)) * CM_ZTAB_W + 1 + col];
      }
      u[n] = a.Q[v * a.stride + idx] - r;
    }
    __syncthreads();
    for (int n = threadIdx.x; n < Np; n += blockDim.x) {
      const int i = n % Nq, jk = n / Nq;
      double t = 0.0; for (int m = 0; m < Nq; ++m) t += a.F[i][m] * u[m + Nq * jk];
      w[n] = t;
    }
    __syncthreads();
    for (int n = threadIdx.x; n < Np; n += blockDim.x) {
      const int i = n % Nq, j = (n / Nq) % Nq, k = n / (Nq * Nq);
      double t = 0.0; for (int m = 0; m < Nq; ++m) t += a.F[j][m] * w[i + Nq * (m + Nq * k)];
      u[n] = t;
    }
    __syncthreads();
    for (int n = threadIdx.x; n < Np; n += blockDim.x) {
      const int ij = n % (Nq * Nq), k = n / (Nq * Nq);
      double t = 0.0; for (int m = 0; m < Nq; ++m) t += a.F[k][m] * u[ij + Nq * Nq * m];
      const long long idx = e * Np + n;
      double r = 0.0;
      if (a.use_ref && (v == 0 || v >= 4)) {
        const int col = (v == 0) ? 0 : (v == 4) ? 1 : 2;
        r = a.general ? a.ref[col * a.stride + idx] : a.ztab[(long long)(a.erow[e] + k) * CM_ZTAB_W + 1 + col];
      }
      a.Q[v * a.stride + idx] = r + t;
    }
    __syncthreads();
  }
}

// a6, second stage: the per-element partial sums are reduced on the device in a fixed order (thread t takes elements
// t, t + T, ...; then a fixed tree), so only 7 doubles travel to the host
__global__ void diag_reduce_kernel(long long n, long long chunk, const double* __restrict__ part, double* __restrict__ out) {
  __shared__ double sh[7][256];
  double r[7] = {0, 0, 0, 0, 0, 0, 0};
  const long long e0 = blockIdx.x * chunk, e1 = (e0 + chunk < n) ? e0 + chunk : n;    // block b reduces entries [e0, e1)
  out += 7 * blockIdx.x;
  for (long long e = e0 + threadIdx.x; e < e1; e += blockDim.x)
    for (int m = 0; m < 7; ++m) { const double v = part[7 * e + m]; r[m] = (m == 5) ? fmax(r[m], v) : r[m] + v; }
  for (int m = 0; m < 7; ++m) sh[m][threadIdx.x] = r[m];
  __syncthreads();
  for (int s = blockDim.x / 2; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s)
      for (int m = 0; m < 7; ++m) sh[m][threadIdx.x] = (m == 5) ? fmax(sh[m][threadIdx.x], sh[m][threadIdx.x + s]) : sh[m][threadIdx.x] + sh[m][threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x < 7) out[threadIdx.x] = sh[threadIdx.x][0];
}

// App. B statistics (eq. B1-B4).  pass 0: per element and nodal zeta-plane the sums of W [1, z, rho, rho phi_m];
// pass 1: of W rho [w' phi'_m, phi'_m^2] with the level means of pass 0.  W = w_i w_j |Ja^3|.
struct ProfArgs {
  int Nq, Np, nvar, general, pass, satadj;
  long long Ne, stride;
  const double* Q; const double* geo; const int* erow; const double* ztab;
  const double* lev;                 // pass 1: [nlev][CM_DG_NPROF] level means
  double A3flat, grav; double w[CM_MAXNQ];
  CmThermo th;
};
constexpr int PROF_NS0 = 9, PROF_NS1 = 12;

__device__ inline void prof_vars(const ProfArgs& a, const double* Y, double Phi, double* phi) {
  const CmThermo& th = a.th;
  const double ir = 1.0 / Y[0];
  const double u = Y[1] * ir, v = Y[2] * ir, w = Y[3] * ir;
  const double rq = (a.nvar == 6) ? Y[5] : 0.0, q = rq * ir;
  const double K = 0.5 * (Y[1] * u + Y[2] * v + Y[3] * w);
  const double kappa = (th.R_d + th.a * q) / (th.c_vd + th.b * q);
  const double E = Y[4] - K - Y[0] * Phi - rq * th.I_v0;
  double pr = kappa * E + th.T_0 * (th.R_d * Y[0] + th.a * rq);
  if (a.satadj) { double Rm, cvm; pr = cm_sat_pressure(th, Y[0], (Y[4] - K) * ir - Phi, q, Rm, cvm); }
  phi[0] = u; phi[1] = v; phi[2] = w; phi[3] = (Y[4] + pr) * ir; phi[4] = q;
  phi[5] = pr * ir * th.iRd * pow(th.p_0 / pr, th.kap_pd);          // theta_v without condensate (R25)
}

__global__ void prof_kernel(const __grid_constant__ ProfArgs a, double* __restrict__ part) {
  extern __shared__ double sh[];                                     // [NF][ns]
  const long long e = blockIdx.x;
  const int Nq = a.Nq, NF = Nq * Nq, ns = a.pass ? PROF_NS1 : PROF_NS0;
  const int ez_row = a.erow[e];                                      // ez * Nq
  for (int k = 0; k < Nq; ++k) {
    for (int m = threadIdx.x; m < NF; m += blockDim.x) {
      const int n = m + NF * k, i = m % Nq, j = m / Nq;
      const long long idx = e * a.Np + n;
      double Y[6] = {0, 0, 0, 0, 0, 0};
      for (int v = 0; v < a.nvar; ++v) Y[v] = a.Q[v * a.stride + idx];
      double z, A3;
      if (a.general) {
        z = a.geo[10 * a.stride + idx];
        const double a0 = a.geo[6 * a.stride + idx], a1 = a.geo[7 * a.stride + idx], a2 = a.geo[8 * a.stride + idx];
        A3 = sqrt(a0 * a0 + a1 * a1 + a2 * a2);
      } else {
        z = 0.0;                                                      // flat: the level height is known in closed form
        A3 = a.A3flat;
      }
      const double Phi = a.general ? a.grav * z : a.ztab[(long long)(ez_row + k) * CM_ZTAB_W];
      const double W = a.w[i] * a.w[j] * A3;
      double phi[6]; prof_vars(a, Y, Phi, phi);
      double* o = sh + m * ns;
      if (a.pass == 0) {
        o[0] = W; o[1] = W * z; o[2] = W * Y[0];
        for (int q = 0; q < 6; ++q) o[3 + q] = W * Y[0] * phi[q];
      } else {
        const double* L = a.lev + (long long)(ez_row + k) * CM_DG_NPROF;
        const double wp = phi[2] - L[2 + 2];
        for (int q = 0; q < 6; ++q) {
          const double fp = phi[q] - L[2 + q];
          o[q] = W * Y[0] * wp * fp; o[6 + q] = W * Y[0] * fp * fp;
        }
      }
    }
    __syncthreads();
    if ((int)threadIdx.x < ns) {
      double s = 0.0;
      for (int m = 0; m < NF; ++m) s += sh[m * ns + threadIdx.x];
      part[(e * Nq + k) * ns + threadIdx.x] = s;
    }
    __syncthreads();
  }
}

// one CTA per level: sums the partials of the Ex*Ey elements of the layer in a fixed order, then normalises
struct ProfRedArgs { int Nq, pass, Ex, Ey, Ez, L, PY, NXC; double flat_dz0, flat_lo, flat_h; int flat_z; double xi[CM_MAXNQ]; };

__global__ void prof_reduce_kernel(const __grid_constant__ ProfRedArgs a, const double* __restrict__ part, double* __restrict__ lev,
                                   double* __restrict__ sumW) {
  __shared__ double sh[PROF_NS1][256];
  const int l = blockIdx.x, ez = l / a.Nq, k = l - ez * a.Nq, ns = a.pass ? PROF_NS1 : PROF_NS0;
  double r[PROF_NS1];
  for (int q = 0; q < PROF_NS1; ++q) r[q] = 0.0;
  for (int h = threadIdx.x; h < a.Ex * a.Ey; h += blockDim.x) {
    const int ex = h % a.Ex, ey = h / a.Ex;
    const long long e = ((((long long)(ey / a.PY) * a.NXC + ex / a.L) * a.Ez + ez) * a.PY + ey % a.PY) * a.L + ex % a.L;
    const double* p = part + (e * a.Nq + k) * ns;
    for (int q = 0; q < ns; ++q) r[q] += p[q];
  }
  for (int q = 0; q < ns; ++q) sh[q][threadIdx.x] = r[q];
  __syncthreads();
  for (int s = blockDim.x / 2; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s) for (int q = 0; q < ns; ++q) sh[q][threadIdx.x] += sh[q][threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    double* o = lev + (long long)l * CM_DG_NPROF;
    if (a.pass == 0) {
      const double sw = sh[0][0];
      sumW[l] = sw;
      o[0] = a.flat_z ? a.flat_lo + (ez + 0.5 * (a.xi[k] + 1.0)) * a.flat_h : sh[1][0] / sw;
      o[1] = sh[2][0] / sw;
      for (int q = 0; q < 6; ++q) o[2 + q] = (sh[3 + q][0] / sw) / o[1];        // (B1)
    } else {
      const double sw = sumW[l];
      for (int q = 0; q < 12; ++q) o[8 + q] = (sh[q][0] / sw) / o[1];           // (B2), (B4)
    }
  }
}

}  // namespace

struct cm_dg_ctx {
  cm_dg_params prm;
  int N, Nq, Np, nvar, ngrad, general, moist;
  int variant = 10;  // 10: row-sweep kernels (cm_dg_kernels10.cuh; flat bricks); 7: CTA-per-element kernels (cm_dg_kernels7.cuh; flat bricks);
                     // 11: CTA-per-element tendency kernel for stored-metric meshes (cm_dg_kernels11.cuh) + thread-per-node gradient;
                     // 2: thread-per-node kernels (cm_dg_kernels2.cuh; any geometry); cm_dg_tuning::kernel selects
  int64_t Ne, stride;
  cudaStream_t st;
  int device = 0;      // the CUDA device the ctx was set up on: every entry point rejects calls made from another one
  std::vector<int32_t> lex_of_elem;
  double xi[CM_MAXNQ], w[CM_MAXNQ], D[CM_MAXNQ][CM_MAXNQ], Filt[CM_MAXNQ][CM_MAXNQ];
  double h[3], min_node_dx;
  size_t em_bytes_per_field = 0;   // bytes per field of G and of the residual (field-major or element-major layout)
  // device
  int *d_nbr = nullptr, *d_erow = nullptr, *d_lex = nullptr;
  double *d_ztab = nullptr, *d_geo = nullptr, *d_ref = nullptr, *d_G = nullptr, *d_res = nullptr, *d_Q2 = nullptr, *d_Q3 = nullptr;
  double *d_zsfc = nullptr, *d_xyz_user = nullptr, *d_part = nullptr, *d_stage = nullptr;
  double *d_lev = nullptr;         // [Ez*Nq][CM_DG_NPROF] level statistics + [Ez*Nq] sum of weights + 8 reduced diagnostics + [256][7] block results
  int tileL = 1, tilePY = 1;       // the tiled element order (x-chunk, y-patch)
  // one time step as a CUDA graph: captured on the second consecutive call with the same state array, dt and coefficient
  // table, replayed afterwards (the 10-12 launches of a step are launch-bound on small meshes)
  // the key holds the coefficient table itself: A_s, B_s and dt are baked into the captured kernel arguments, so two tables
  // may share a graph only if every entry is equal (a checksum could collide and replay stale coefficients silently)
  struct StepKey {
    const double* Q = nullptr; double dt = 0.0; int nstages = 0; std::vector<double> A, B;
    bool operator==(const StepKey& o) const { return Q == o.Q && dt == o.dt && nstages == o.nstages && A == o.A && B == o.B; }
  };
  bool graphs = true;
  cudaGraphExec_t step_exec = nullptr;
  StepKey step_key, last_key;
  CmKP kp;
  cm_launch_fn launch_grad = nullptr, launch_tend = nullptr;
  int ahead_t = -1, ahead_g = -1;   // L2 prefetch distance of the tendency / gradient kernel (-1 = one wave)
  // profiling
  bool profiling = false;
  std::vector<cudaEvent_t> ev;   // pairs (start, stop)
  std::vector<int> ev_kind;      // per pair: 0 gradient, 1 tendency, 2 other
  size_t ev_used = 0;
};

namespace {

void free_ctx(cm_dg_ctx* c) {
  if (!c) return;
  cudaFree(c->d_nbr); cudaFree(c->d_erow); cudaFree(c->d_lex); cudaFree(c->d_ztab); cudaFree(c->d_geo);
  cudaFree(c->d_ref); cudaFree(c->d_G); cudaFree(c->d_res); cudaFree(c->d_Q2); cudaFree(c->d_Q3); cudaFree(c->d_zsfc);
  cudaFree(c->d_xyz_user); cudaFree(c->d_part); cudaFree(c->d_stage); cudaFree(c->d_lev);
  for (auto e : c->ev) cudaEventDestroy(e);
  if (c->step_exec) cudaGraphExecDestroy(c->step_exec);
  delete c;
}

// Every computing entry point starts here: the ctx is bound to the device that was current in cm_dg_setup.
int enter(const cm_dg_ctx* c, const char* who) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return fail(CM_DG_ECUDA, std::string(who) + ": cudaGetDevice failed");
  if (dev != c->device)
    return fail(CM_DG_ESTATE, std::string(who) + ": the ctx belongs to CUDA device " + std::to_string(c->device) +
                              " but the current device is " + std::to_string(dev));
  return CM_DG_OK;
}

GeoArgs geo_args(const cm_dg_ctx* c) {
  GeoArgs a;
  a.Nq = c->Nq; a.Np = c->Np; a.geom = c->prm.geom; a.Ne = c->Ne; a.stride = c->stride;
  for (int d = 0; d < 3; ++d) { a.ne[d] = c->prm.ne[d]; a.lo[d] = c->prm.lo[d]; a.hi[d] = c->prm.hi[d]; a.h[d] = c->h[d]; }
  a.lex = c->d_lex; a.zsfc = c->d_zsfc; a.xyz_user = c->d_xyz_user;
  for (int i = 0; i < CM_MAXNQ; ++i) { a.xi[i] = c->xi[i]; a.w[i] = c->w[i]; for (int j = 0; j < CM_MAXNQ; ++j) a.D[i][j] = c->D[i][j]; }
  a.cs = c->prm.C_s; a.grav = c->prm.grav;
  a.N = c->N; a.metric_form = c->prm.metric_form;
  a.sp_alpha = c->prm.sponge_alpha; a.sp_zs = c->prm.sponge_zs; a.sp_gamma = c->prm.sponge_gamma;
  return a;
}

// timed launch helper
struct Timed {
  cm_dg_ctx* c; int kind; bool on;
  Timed(cm_dg_ctx* c_, int kind_) : c(c_), kind(kind_), on(c_->profiling) {
    if (!on) return;
    if (c->ev_used + 2 > c->ev.size()) {
      for (int t = 0; t < 2; ++t) { cudaEvent_t e; cudaEventCreate(&e); c->ev.push_back(e); }
      c->ev_kind.push_back(kind);
    }
    c->ev_kind[c->ev_used / 2] = kind;
    cudaEventRecord(c->ev[c->ev_used], c->st);
  }
  ~Timed() {
    if (!on) return;
    cudaEventRecord(c->ev[c->ev_used + 1], c->st);
    c->ev_used += 2;
  }
};

bool misaligned(const void* ptr) { return (reinterpret_cast<uintptr_t>(ptr) & 15u) != 0; }

int run_gradient(cm_dg_ctx* c, const double* Q, double* Gout, int raw) {
  if (misaligned(Q) || misaligned(Gout)) return fail(CM_DG_EINVAL, "state arrays must be 16-byte aligned (bulk TMA source)");
  CmKP kp = c->kp;
  kp.Q = Q; kp.Gout = Gout; kp.mode = raw; kp.ahead = c->ahead_g;
  Timed t(c, 0);
  cudaError_t err = c->launch_grad(kp, c->moist, c->general, c->variant, c->st);
  if (err != cudaSuccess) return fail(CM_DG_ECUDA, std::string("gradient kernel launch: ") + cudaGetErrorString(err));
  return CM_DG_OK;
}

int run_tendency(cm_dg_ctx* c, const double* Q, double* dQ, double* Qnew, int mode, double rka, double rkb, double dt) {
  if (misaligned(Q) || misaligned(dQ) || misaligned(Qnew)) return fail(CM_DG_EINVAL, "state arrays must be 16-byte aligned (bulk TMA source)");
  CmKP kp = c->kp;
  kp.ahead = c->ahead_t;
  kp.Q = Q; kp.G = c->d_G; kp.dQ = dQ; kp.Qnew = Qnew; kp.mode = mode; kp.rka = rka; kp.rkb = rkb; kp.dt = dt;
  Timed t(c, 1);
  cudaError_t err = c->launch_tend(kp, c->moist, c->general, c->variant, c->st);
  if (err != cudaSuccess) return fail(CM_DG_ECUDA, std::string("tendency kernel launch: ") + cudaGetErrorString(err));
  return CM_DG_OK;
}

}  // namespace

extern "C" {

const char* cm_dg_last_error(void) { return g_err.c_str(); }

void cm_dg_destroy(cm_dg_ctx* ctx) { free_ctx(ctx); }

int cm_dg_setup(const cm_dg_params* p, void* cuda_stream, cm_dg_ctx** out) {
  return cm_dg_setup_tuned(p, nullptr, cuda_stream, out);
}

int cm_dg_setup_tuned(const cm_dg_params* p, const cm_dg_tuning* tune, void* cuda_stream, cm_dg_ctx** out) {
  if (!p || !out) return fail(CM_DG_EINVAL, "cm_dg_setup: NULL argument");
  *out = nullptr;   // before the first early return: a refused setup never leaves a stale handle behind
  cm_dg_tuning tn;
  std::memset(&tn, 0, sizeof(tn));
  tn.ahead_t = tn.ahead_g = -1;
  if (tune) tn = *tune;
  if (tn.kernel != 0 && tn.kernel != 2 && tn.kernel != 7 && tn.kernel != 10 && tn.kernel != 11) return fail(CM_DG_EINVAL, "cm_dg_setup_tuned: kernel must be 0, 2, 7, 10 or 11");
  if (tn.max_chunk < 0 || tn.max_patch < 0 || tn.row_len < 0) return fail(CM_DG_EINVAL, "cm_dg_setup_tuned: negative tile size");
  if (p->N < 2 || p->N > 7) return fail(CM_DG_EINVAL, "cm_dg_setup: polynomial order N must be in 2..7");
  if (p->nvar != 5 && p->nvar != 6) return fail(CM_DG_EINVAL, "cm_dg_setup: nvar must be 5 or 6");
  for (int d = 0; d < 3; ++d) {
    if (p->ne[d] < 1) return fail(CM_DG_EINVAL, "cm_dg_setup: ne[d] must be >= 1");
    if (!(p->hi[d] > p->lo[d])) return fail(CM_DG_EINVAL, "cm_dg_setup: hi[d] must exceed lo[d]");
    if (p->bc[d] != 0 && p->bc[d] != 1) return fail(CM_DG_EINVAL, "cm_dg_setup: bc[d] must be 0 (periodic) or 1 (wall)");
  }
  if (p->geom < 0 || p->geom > 2) return fail(CM_DG_EINVAL, "cm_dg_setup: geom must be 0, 1 or 2");
  if (p->geom == 1 && !p->zsfc_nodes) return fail(CM_DG_EINVAL, "cm_dg_setup: geom == 1 needs zsfc_nodes");
  if (p->geom == 2 && !p->xyz) return fail(CM_DG_EINVAL, "cm_dg_setup: geom == 2 needs xyz");
  if (p->use_ref && (!p->ref_rho || !p->ref_rhoe || (p->nvar == 6 && !p->ref_rhoq)))
    return fail(CM_DG_EINVAL, "cm_dg_setup: use_ref needs ref_rho, ref_rhoe (and ref_rhoq when nvar == 6)");
  if (p->sgs < 0 || p->sgs > 2) return fail(CM_DG_EINVAL, "cm_dg_setup: sgs must be 0 (inviscid), 1 (Smagorinsky-Lilly) or 2 (Vreman)");
  if (p->sgs && !(p->Pr_t > 0.0)) return fail(CM_DG_EINVAL, "cm_dg_setup: Pr_t must be positive");
  if (p->richardson != 0 && p->richardson != 1) return fail(CM_DG_EINVAL, "cm_dg_setup: richardson must be 0 or 1");
  if (p->richardson && !p->sgs) return fail(CM_DG_EINVAL, "cm_dg_setup: richardson = 1 needs an eddy-viscosity closure (sgs != 0)");
  if (p->p_0 < 0.0) return fail(CM_DG_EINVAL, "cm_dg_setup: p_0 must be positive (0 = 1e5 Pa)");
  if (p->riemann < 0 || p->riemann > 2) return fail(CM_DG_EINVAL, "cm_dg_setup: riemann must be 0 (Rusanov), 1 (HLLC) or 2 (Roe)");
  if (p->metric_form != 0 && p->metric_form != 1) return fail(CM_DG_EINVAL, "cm_dg_setup: metric_form must be 0 or 1");
  if (p->filter_order < 0 || p->filter_alpha < 0.0) return fail(CM_DG_EINVAL, "cm_dg_setup: filter_order and filter_alpha must be >= 0");
  if (p->sponge_alpha < 0.0 || p->sponge_gamma < 0) return fail(CM_DG_EINVAL, "cm_dg_setup: sponge_alpha and sponge_gamma must be >= 0");
  if (p->sponge_alpha > 0.0 && !(p->sponge_zs < p->hi[2])) return fail(CM_DG_EINVAL, "cm_dg_setup: the sponge must start below hi[2]");
  if (!(p->c_vd > 0.0) || !(p->R_d > 0.0)) return fail(CM_DG_EINVAL, "cm_dg_setup: R_d and c_vd must be positive");
  if (p->satadj != 0 && p->satadj != 1) return fail(CM_DG_EINVAL, "cm_dg_setup: satadj must be 0 or 1");
  if (p->satadj && p->nvar != 6) return fail(CM_DG_EINVAL, "cm_dg_setup: satadj = 1 needs the moisture tracer (nvar == 6)");
  if (p->c_vl < 0.0 || p->p_triple < 0.0 || p->T_triple < 0.0) return fail(CM_DG_EINVAL, "cm_dg_setup: c_vl, p_triple, T_triple must be >= 0");
  if (p->drag_cd < 0.0) return fail(CM_DG_EINVAL, "cm_dg_setup: drag_cd must be >= 0");
  if ((p->drag_cd != 0.0 || p->lhf_bottom != 0.0 || p->evap_bottom != 0.0) && p->bc[2] != 1)
    return fail(CM_DG_EINVAL, "cm_dg_setup: surface fluxes (drag_cd, lhf_bottom, evap_bottom) need a wall in z (bc[2] == 1)");
  if (p->evap_bottom != 0.0 && p->nvar != 6)
    return fail(CM_DG_EINVAL, "cm_dg_setup: evap_bottom needs the moisture tracer (nvar == 6): a dry run would drop the prescribed mass and water flux");
  const int64_t Ne = (int64_t)p->ne[0] * p->ne[1] * p->ne[2];
  const int Nq = p->N + 1, Np = Nq * Nq * Nq;
  if (Ne * Np >= (int64_t)1 << 31) return fail(CM_DG_EINVAL, "cm_dg_setup: more than 2^31 nodes");

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
    return fail(CM_DG_ECUDA, "cm_dg_setup: no CUDA device (this library has no CPU path)");

  cm_dg_ctx* c = new cm_dg_ctx();
  c->prm = *p;
  c->prm.zsfc_nodes = nullptr; c->prm.xyz = nullptr; c->prm.ref_rho = c->prm.ref_rhoe = c->prm.ref_rhoq = nullptr;
  if (c->prm.p_0 == 0.0) c->prm.p_0 = 1.0e5;
  if (c->prm.sponge_gamma == 0) c->prm.sponge_gamma = 2;
  if (c->prm.filter_alpha == 0.0) c->prm.filter_alpha = 36.0436533891172;   // -log(2^-52)
  c->N = p->N; c->Nq = Nq; c->Np = Np; c->nvar = p->nvar; c->moist = (p->nvar == 6);
  c->ngrad = c->moist ? 12 : 9;
  c->Ne = Ne;
  c->stride = ((Ne * Np + 1 + 31) / 32) * 32;   // >= Ne*Np + 1: the bulk-TMA tile fetch of the last element reads one double past it
  c->st = (cudaStream_t)cuda_stream;
  if (cudaGetDevice(&c->device) != cudaSuccess) { delete c; return fail(CM_DG_ECUDA, "cm_dg_setup: cudaGetDevice failed"); }
  for (int d = 0; d < 3; ++d) c->h[d] = (p->hi[d] - p->lo[d]) / p->ne[d];
  std::memset(c->D, 0, sizeof(c->D));
  lgl_operators(c->N, c->xi, c->w, c->D);
  std::memset(c->Filt, 0, sizeof(c->Filt));
  if (c->prm.filter_order > 0) filter_operator(c->N, c->xi, c->prm.filter_order, c->prm.filter_alpha, c->Filt);

  // ---- element order (library order = launch order of the CTA-per-element kernels)
  // e = ((((ey / PY) * NXC + ex / L) * Ez + ez) * PY + ey % PY) * L + ex % L with L | Ex, PY | Ey: consecutive CTAs
  // walk up a column of (PY x L)-element tiles, so that the one wave of resident CTAs works on a compact brick and
  // the x/y/z neighbour traces are in L2 when they are gathered (a z neighbour is PY*L elements away, a y/x
  // neighbour at most Ez*PY*L).  The flat kernels recompute this map from blockIdx (cm6_position).
  int L = 1, PY = 1;
  {
    const bool lex_order = tn.order_lex != 0;
    const int maxL = tn.max_chunk > 0 ? tn.max_chunk : 32, maxPY = tn.max_patch > 0 ? tn.max_patch : 16;
    for (int d = 1; d <= p->ne[0] && d <= maxL; ++d) if (p->ne[0] % d == 0) L = d;
    for (int d = 1; d <= p->ne[1] && d <= maxPY; ++d) if (p->ne[1] % d == 0) PY = d;
    if (lex_order) { L = p->ne[0]; PY = p->ne[1]; }
    c->lex_of_elem.resize(Ne);
    const int NXC = p->ne[0] / L;
    for (int64_t l = 0; l < Ne; ++l) {
      const int64_t ex = l % p->ne[0], ey = (l / p->ne[0]) % p->ne[1], ez = l / ((int64_t)p->ne[0] * p->ne[1]);
      const int64_t e = ((((ey / PY) * NXC + ex / L) * p->ne[2] + ez) * PY + ey % PY) * L + ex % L;
      c->lex_of_elem[e] = (int32_t)l;
    }
  }
  std::vector<int32_t> pos_of_lex(Ne);
  for (int64_t e = 0; e < Ne; ++e) pos_of_lex[c->lex_of_elem[e]] = (int32_t)e;

  // ---- connectivity: faces 0..5 = -xi, +xi, -eta, +eta, -zeta, +zeta; -1 = wall
  std::vector<int32_t> nbr(Ne * 6), erow(Ne);
  for (int64_t e = 0; e < Ne; ++e) {
    const int64_t l = c->lex_of_elem[e];
    int ec[3] = {(int)(l % p->ne[0]), (int)((l / p->ne[0]) % p->ne[1]), (int)(l / ((int64_t)p->ne[0] * p->ne[1]))};
    erow[e] = ec[2] * Nq;
    for (int f = 0; f < 6; ++f) {
      const int d = f / 2;
      int v[3] = {ec[0], ec[1], ec[2]};
      v[d] += (f % 2) ? 1 : -1;
      if (v[d] < 0 || v[d] >= p->ne[d]) {
        if (p->bc[d] == 1) { nbr[e * 6 + f] = -1; continue; }
        v[d] = (v[d] + p->ne[d]) % p->ne[d];
      }
      nbr[e * 6 + f] = pos_of_lex[v[0] + (int64_t)p->ne[0] * (v[1] + (int64_t)p->ne[1] * v[2])];
    }
  }

  // ---- reference state: z-only table on flat meshes, per-node arrays otherwise
  const size_t nn = (size_t)Ne * Np;
  bool ref_z_only = true;
  if (p->use_ref && p->geom == 0) {
    const int64_t nh = (int64_t)p->ne[0] * p->ne[1];
    for (int ez = 0; ez < p->ne[2] && ref_z_only; ++ez)
      for (int k = 0; k < Nq && ref_z_only; ++k) {
        const size_t first = ((size_t)ez * nh) * Np + (size_t)k * Nq * Nq;
        for (int64_t hh = 0; hh < nh && ref_z_only; ++hh)
          for (int m = 0; m < Nq * Nq; ++m) {
            const size_t id = ((size_t)ez * nh + hh) * Np + (size_t)k * Nq * Nq + m;
            if (p->ref_rho[id] != p->ref_rho[first] || p->ref_rhoe[id] != p->ref_rhoe[first] ||
                (c->moist && p->ref_rhoq[id] != p->ref_rhoq[first])) { ref_z_only = false; break; }
          }
      }
  }
  c->general = (p->geom != 0 || (p->use_ref && !ref_z_only) || p->metric_form == 1) ? 1 : 0;
  if (tn.force_general) c->general = 1;
  if (tn.kernel) c->variant = tn.kernel;
  // stored-metric meshes: CTA-per-element tendency kernel fed by bulk TMA (cm_dg_kernels11.cuh) with the thread-per-node
  // gradient kernel; kernel = 2 keeps the thread-per-node tendency kernel as well
  if (c->general) c->variant = (tn.kernel == 2) ? 2 : 11;
  // HLLC, Roe and the saturation adjustment are implemented in the thread-per-node kernels; so is the Richardson factor at
  // the orders whose flat gradient kernel is the trace-buffer one (N <= 3)
  if (p->riemann != 0 || p->satadj || (!c->general && p->richardson && Nq <= 4)) c->variant = 2;

  auto bail = [&](int code) { free_ctx(c); return code; };
#define CM_CUDA_B(call)                                                                                   \
  do {                                                                                                    \
    cudaError_t err__ = (call);                                                                           \
    if (err__ != cudaSuccess) {                                                                           \
      fail(err__ == cudaErrorMemoryAllocation ? CM_DG_ENOMEM : CM_DG_ECUDA, std::string(#call) + ": " + cudaGetErrorString(err__)); \
      return bail(err__ == cudaErrorMemoryAllocation ? CM_DG_ENOMEM : CM_DG_ECUDA);                       \
    }                                                                                                     \
  } while (0)

  const size_t fbytes = (size_t)c->stride * sizeof(double);
  CM_CUDA_B(cudaMalloc(&c->d_nbr, nbr.size() * sizeof(int32_t)));
  CM_CUDA_B(cudaMalloc(&c->d_erow, erow.size() * sizeof(int32_t)));
  CM_CUDA_B(cudaMalloc(&c->d_lex, (size_t)Ne * sizeof(int32_t)));
  CM_CUDA_B(cudaMemcpy(c->d_nbr, nbr.data(), nbr.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
  CM_CUDA_B(cudaMemcpy(c->d_erow, erow.data(), erow.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
  CM_CUDA_B(cudaMemcpy(c->d_lex, c->lex_of_elem.data(), (size_t)Ne * sizeof(int32_t), cudaMemcpyHostToDevice));
  if (p->geom == 1) {
    const size_t nz = (size_t)p->ne[0] * Nq * p->ne[1] * Nq;
    CM_CUDA_B(cudaMalloc(&c->d_zsfc, nz * sizeof(double)));
    CM_CUDA_B(cudaMemcpy(c->d_zsfc, p->zsfc_nodes, nz * sizeof(double), cudaMemcpyHostToDevice));
  }
  if (p->geom == 2) {
    std::vector<double> tmp((size_t)3 * c->stride, 0.0);
    for (int d = 0; d < 3; ++d)
      for (int64_t e = 0; e < Ne; ++e)
        std::memcpy(&tmp[(size_t)d * c->stride + (size_t)e * Np], p->xyz + ((size_t)d * Ne + c->lex_of_elem[e]) * Np, Np * sizeof(double));
    CM_CUDA_B(cudaMalloc(&c->d_xyz_user, tmp.size() * sizeof(double)));
    CM_CUDA_B(cudaMemcpy(c->d_xyz_user, tmp.data(), tmp.size() * sizeof(double), cudaMemcpyHostToDevice));
  }

  // ---- kernel parameter block
  CmKP& kp = c->kp;
  std::memset(&kp, 0, sizeof(kp));
  kp.ginvL = 1.0f / (float)L; kp.ginvNXC = 1.0f / (float)(p->ne[0] / L);
  kp.gL = L; kp.gPY = PY; kp.gNXC = p->ne[0] / L; kp.gNYP = p->ne[1] / PY; kp.gEz = p->ne[2];
  c->tileL = L; c->tilePY = PY;
  for (int d = 0; d < 3; ++d) kp.gbc[d] = p->bc[d];
  kp.ahead = -1;   // L2 prefetch distance of the cm7 kernels: -1 = one wave of resident CTAs (set by the launcher)
  c->ahead_t = tn.ahead_t; c->ahead_g = tn.ahead_g;
  c->graphs = tn.no_graph == 0;
  kp.gS = L;       // row-sweep kernels: a row is a whole x-chunk unless the mesh is small or the tuning asks for shorter rows
  {
    // small meshes: long rows leave too few CTAs for an even last wave (config 3 at 32x32x16: 512 rows of 32 on 444 CTA
    // slots, 7.1 G DOF-stages/s; rows of 8: 8.6 G).  Longest row that still gives >= 4 waves of 3 CTAs per SM, but not
    // below 8 elements (the pipeline fill of a row is one element)
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device);
    const int64_t want = (int64_t)4 * 3 * sms;
    int best = 0;
    for (int S = L; S >= 1; --S) if (L % S == 0 && Ne / S >= want) { best = S; break; }
    if (best < 8) { best = L; for (int S = 8; S <= L; ++S) if (L % S == 0) { best = S; break; } }
    kp.gS = best;
  }
  if (tn.row_len > 0) {
    if (L % tn.row_len != 0) { fail(CM_DG_EINVAL, "cm_dg_setup_tuned: row_len must divide the x-chunk length"); return bail(CM_DG_EINVAL); }
    kp.gS = tn.row_len;
  }
  if (c->variant == 11 && (p->ne[2] > 65535 || (int64_t)kp.gNXC * kp.gNYP > 65535)) c->variant = 2;   // 1-D grid instead
  if (c->variant != 2 && ((int64_t)PY * L > 2147483647LL || p->ne[2] > 65535 || (int64_t)kp.gNXC * kp.gNYP > 65535)) {   // 3-D grid of the flat kernels
    fail(CM_DG_EINVAL, "cm_dg_setup: mesh exceeds the launch-grid limits (Ez and (Ex/L)*(Ey/PY) must be <= 65535)");
    return bail(CM_DG_EINVAL);
  }
  kp.Ne = (int)Ne; kp.stride = c->stride; kp.sgs = p->sgs; kp.use_ref = p->use_ref ? 1 : 0;
  kp.richardson = p->richardson; kp.riemann = p->riemann;
  kp.terrain = (p->geom == 1 && p->metric_form == 0 && !tn.no_terrain) ? 1 : 0;
  kp.cs2 = p->C_s * p->C_s;
  for (int d = 0; d < 3; ++d) { kp.d2[d] = (c->h[d] / c->N) * (c->h[d] / c->N); kp.urelax[d] = p->u_relax[d]; }
  kp.th.p_0 = c->prm.p_0; kp.th.kap_pd = p->R_d / (p->c_vd + p->R_d); kp.th.iRd = 1.0 / p->R_d;
  kp.th.R_d = p->R_d; kp.th.c_vd = p->c_vd; kp.th.a = p->R_v - p->R_d; kp.th.b = p->c_vv - p->c_vd;
  kp.th.T_0 = p->T_0; kp.th.I_v0 = p->I_v0; kp.th.grav = p->grav;
  kp.th.dk = kp.th.a * p->c_vd - p->R_d * kp.th.b;
  kp.th.icvd = 1.0 / p->c_vd; kp.th.kappa_d = p->R_d / p->c_vd;
  {
    const double c_vl = p->c_vl > 0.0 ? p->c_vl : 4181.0, p_tr = p->p_triple > 0.0 ? p->p_triple : 611.657;
    const double T_tr = p->T_triple > 0.0 ? p->T_triple : 273.16;
    kp.satadj = p->satadj;
    kp.th.R_v = p->R_v; kp.th.c_vv = p->c_vv; kp.th.c_vl = c_vl;
    kp.th.Lv0 = p->I_v0 + p->R_v * p->T_0;                                 // eq. (9)
    kp.th.dcp = p->c_vv + p->R_v - c_vl;
    kp.th.p_tr = p_tr; kp.th.iT_tr = 1.0 / T_tr;
    kp.th.sx1 = kp.th.dcp / p->R_v; kp.th.sx2 = (kp.th.Lv0 - kp.th.dcp * p->T_0) / p->R_v;
  }
  kp.cA[0] = c->h[1] * c->h[2] / 4.0; kp.cA[1] = c->h[0] * c->h[2] / 4.0; kp.cA[2] = c->h[0] * c->h[1] / 4.0;
  kp.invJ = 8.0 / (c->h[0] * c->h[1] * c->h[2]);
  {
    const double delta = std::cbrt(c->h[0] * c->h[1] * c->h[2]) / c->N;
    kp.cs2delta2 = (p->C_s * delta) * (p->C_s * delta);
  }
  kp.inv_Pr = p->sgs ? 1.0 / p->Pr_t : 0.0;
  kp.shf = p->shf_bottom + p->lhf_bottom;   // n_in . rho (J + D) = SHF + LHF
  kp.evap = p->evap_bottom; kp.drag_cd = p->drag_cd;
  kp.inv_w0 = 1.0 / c->w[0];
  for (int i = 0; i < CM_MAXNQ; ++i) for (int j = 0; j < CM_MAXNQ; ++j) kp.D[i][j] = c->D[i][j];
  kp.nbr = c->d_nbr; kp.erow = c->d_erow;

  c->min_node_dx = std::min(c->h[0], std::min(c->h[1], c->h[2])) * 0.5 * (c->xi[1] - c->xi[0]);

  if (!c->general) {
    // z table: Phi and the reference column per (ez, k)
    const int rows = p->ne[2] * Nq;
    std::vector<double> zt((size_t)rows * CM_ZTAB_W, 0.0);
    const int64_t nh = (int64_t)p->ne[0] * p->ne[1];
    for (int ez = 0; ez < p->ne[2]; ++ez)
      for (int k = 0; k < Nq; ++k) {
        double* t = &zt[(size_t)(ez * Nq + k) * CM_ZTAB_W];
        const double z = p->lo[2] + (ez + 0.5 * (c->xi[k] + 1.0)) * c->h[2];
        t[0] = p->grav * z;
        t[7] = 0.0;                                                        // Rayleigh sponge coefficient tau_s(z) (A5, R18)
        if (c->prm.sponge_alpha > 0.0 && z > c->prm.sponge_zs)
          t[7] = c->prm.sponge_alpha *
                 std::pow(std::sin(0.5 * 3.14159265358979323846 * (z - c->prm.sponge_zs) / (p->hi[2] - c->prm.sponge_zs)), (double)c->prm.sponge_gamma);
        if (p->use_ref) {
          const size_t id = ((size_t)ez * nh) * Np + (size_t)k * Nq * Nq;
          t[1] = p->ref_rho[id]; t[2] = p->ref_rhoe[id]; t[3] = c->moist ? p->ref_rhoq[id] : 0.0;
          t[4] = t[2] - t[1] * t[0] - t[3] * p->I_v0;
          t[5] = t[3] / t[1];
          t[6] = 1.0 / (p->c_vd + kp.th.b * t[5]);
        }
      }
    CM_CUDA_B(cudaMalloc(&c->d_ztab, zt.size() * sizeof(double)));
    CM_CUDA_B(cudaMemcpy(c->d_ztab, zt.data(), zt.size() * sizeof(double), cudaMemcpyHostToDevice));
    kp.ztab = c->d_ztab;
  } else {
    CM_CUDA_B(cudaMalloc(&c->d_geo, (size_t)CM_NGEO * fbytes));
    CM_CUDA_B(cudaMemset(c->d_geo, 0, (size_t)CM_NGEO * fbytes));
    double* d_chk = nullptr;
    CM_CUDA_B(cudaMalloc(&d_chk, (size_t)Ne * 3 * sizeof(double)));
    GeoArgs ga = geo_args(c);
    const int thr = 128;
    const size_t sm = (size_t)(24 * Np + 4 * thr) * sizeof(double);
    cudaError_t err = cudaFuncSetAttribute(metrics_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (err == cudaSuccess) { metrics_kernel<<<(unsigned)Ne, thr, sm, c->st>>>(ga, c->d_geo, d_chk); err = cudaGetLastError(); }
    std::vector<double> chk((size_t)Ne * 3);
    if (err == cudaSuccess) err = cudaMemcpyAsync(chk.data(), d_chk, chk.size() * sizeof(double), cudaMemcpyDeviceToHost, c->st);
    if (err == cudaSuccess) err = cudaStreamSynchronize(c->st);
    cudaFree(d_chk);
    if (err != cudaSuccess) { fail(CM_DG_ECUDA, std::string("metrics kernel: ") + cudaGetErrorString(err)); return bail(CM_DG_ECUDA); }
    double minJ = 1e300, res = 0, mdx = 1e300;
    for (int64_t e = 0; e < Ne; ++e) { minJ = std::min(minJ, chk[3 * e]); res = std::max(res, chk[3 * e + 1]); mdx = std::min(mdx, chk[3 * e + 2]); }
    if (!(minJ > 0.0)) { fail(CM_DG_EINVAL, "cm_dg_setup: non-positive Jacobian determinant in the mesh"); return bail(CM_DG_EINVAL); }
    if (res > 1e-10) {
      char buf[200]; std::snprintf(buf, sizeof buf, "cm_dg_setup: discrete metric identity violated (%.3e > 1e-10): a fully 3-D warp needs metric_form = 1", res);
      fail(CM_DG_EINVAL, buf); return bail(CM_DG_EINVAL);
    }
    c->min_node_dx = mdx;
    kp.geo = c->d_geo;
    if (p->use_ref) {
      std::vector<double> tmp((size_t)3 * c->stride, 0.0);
      const double* src[3] = {p->ref_rho, p->ref_rhoe, c->moist ? p->ref_rhoq : nullptr};
      for (int a = 0; a < 3; ++a)
        if (src[a])
          for (int64_t e = 0; e < Ne; ++e)
            std::memcpy(&tmp[(size_t)a * c->stride + (size_t)e * Np], src[a] + (size_t)c->lex_of_elem[e] * Np, Np * sizeof(double));
      CM_CUDA_B(cudaMalloc(&c->d_ref, tmp.size() * sizeof(double)));
      CM_CUDA_B(cudaMemcpy(c->d_ref, tmp.data(), tmp.size() * sizeof(double), cudaMemcpyHostToDevice));
      kp.ref = c->d_ref;
    }
  }
  (void)nn;

  // ---- scratch owned by the ctx
  // element-major internal arrays of the row-sweep kernels: [e][field][SLOT], SLOT = Np rounded up to even
  const size_t slot = (size_t)Np + (Np & 1);
  c->em_bytes_per_field = std::max(fbytes, (size_t)Ne * slot * sizeof(double));
  if (p->sgs) CM_CUDA_B(cudaMalloc(&c->d_G, (size_t)c->ngrad * c->em_bytes_per_field));
  CM_CUDA_B(cudaMalloc(&c->d_part, (size_t)Ne * 7 * sizeof(double)));
  CM_CUDA_B(cudaMalloc(&c->d_lev, ((size_t)p->ne[2] * Nq * (CM_DG_NPROF + 1) + 8 + 7 * 256) * sizeof(double)));
  // LSRK residual and the two further state buffers of the stage ring (cm_dg_lsrk_step never allocates or synchronises)
  {
    const size_t sb = (size_t)c->nvar * fbytes;
    CM_CUDA_B(cudaMalloc(&c->d_res, (size_t)c->nvar * c->em_bytes_per_field));
    CM_CUDA_B(cudaMalloc(&c->d_Q2, sb)); CM_CUDA_B(cudaMemsetAsync(c->d_Q2, 0, sb, c->st));
    CM_CUDA_B(cudaMalloc(&c->d_Q3, sb)); CM_CUDA_B(cudaMemsetAsync(c->d_Q3, 0, sb, c->st));
  }

  switch (Nq) {
    case 3: c->launch_grad = cm_launch_gradient_nq3; c->launch_tend = cm_launch_tendency_nq3; break;
    case 4: c->launch_grad = cm_launch_gradient_nq4; c->launch_tend = cm_launch_tendency_nq4; break;
    case 5: c->launch_grad = cm_launch_gradient_nq5; c->launch_tend = cm_launch_tendency_nq5; break;
    case 6: c->launch_grad = cm_launch_gradient_nq6; c->launch_tend = cm_launch_tendency_nq6; break;
    case 7: c->launch_grad = cm_launch_gradient_nq7; c->launch_tend = cm_launch_tendency_nq7; break;
    default: c->launch_grad = cm_launch_gradient_nq8; c->launch_tend = cm_launch_tendency_nq8; break;
  }
  CM_CUDA_B(cudaStreamSynchronize(c->st));
  *out = c;
  return CM_DG_OK;
}

int cm_dg_layout(const cm_dg_ctx* ctx, int64_t* n_elem, int32_t* np, int64_t* field_stride, int32_t* lex_of_elem) {
  if (!ctx) return fail(CM_DG_EINVAL, "cm_dg_layout: NULL ctx");
  if (n_elem) *n_elem = ctx->Ne;
  if (np) *np = ctx->Np;
  if (field_stride) *field_stride = ctx->stride;
  if (lex_of_elem) std::memcpy(lex_of_elem, ctx->lex_of_elem.data(), (size_t)ctx->Ne * sizeof(int32_t));
  return CM_DG_OK;
}

int cm_dg_coords(cm_dg_ctx* ctx, double* xyz_dev) {
  if (!ctx || !xyz_dev) return fail(CM_DG_EINVAL, "cm_dg_coords: NULL argument");
  { int rc_ = enter(ctx, "cm_dg_coords"); if (rc_) return rc_; }
  GeoArgs ga = geo_args(ctx);
  coords_kernel<<<(unsigned)ctx->Ne, 128, 0, ctx->st>>>(ga, xyz_dev);
  CM_CUDA(cudaGetLastError());
  return CM_DG_OK;
}

int cm_dg_metrics(cm_dg_ctx* ctx, double* Ja_dev, double* J_dev) {
  if (!ctx || !Ja_dev || !J_dev) return fail(CM_DG_EINVAL, "cm_dg_metrics: NULL argument");
  { int rc_ = enter(ctx, "cm_dg_metrics"); if (rc_) return rc_; }
  const long long n = ctx->Ne * ctx->Np;
  const int thr = 256; const unsigned blocks = (unsigned)((n + thr - 1) / thr);
  if (ctx->general)
    general_metrics_copy<<<blocks, thr, 0, ctx->st>>>(n, ctx->stride, ctx->d_geo, Ja_dev, J_dev);
  else
    flat_metrics_fill<<<blocks, thr, 0, ctx->st>>>(n, ctx->stride, ctx->kp.cA[0], ctx->kp.cA[1], ctx->kp.cA[2], 1.0 / ctx->kp.invJ, Ja_dev, J_dev);
  CM_CUDA(cudaGetLastError());
  return CM_DG_OK;
}

int cm_dg_gradient(cm_dg_ctx* ctx, const double* Q_dev, double* G_dev) {
  if (!ctx || !Q_dev || !G_dev) return fail(CM_DG_EINVAL, "cm_dg_gradient: NULL argument");
  { int rc_ = enter(ctx, "cm_dg_gradient"); if (rc_) return rc_; }
  return run_gradient(ctx, Q_dev, G_dev, 1);
}

int cm_dg_rhs(cm_dg_ctx* ctx, const double* Q_dev, double* dQ_dev, double t) {
  (void)t;   // no time-dependent forcing on this path (reading R14)
  if (!ctx || !Q_dev || !dQ_dev) return fail(CM_DG_EINVAL, "cm_dg_rhs: NULL argument");
  if (Q_dev == dQ_dev) return fail(CM_DG_EINVAL, "cm_dg_rhs: Q and dQ must be distinct buffers");
  { int rc_ = enter(ctx, "cm_dg_rhs"); if (rc_) return rc_; }
  if (ctx->prm.sgs) { int rc = run_gradient(ctx, Q_dev, ctx->d_G, 0); if (rc) return rc; }
  return run_tendency(ctx, Q_dev, dQ_dev, nullptr, 0, 0.0, 0.0, 0.0);
}

int cm_dg_filter(cm_dg_ctx* ctx, double* Q_dev) {
  if (!ctx || !Q_dev) return fail(CM_DG_EINVAL, "cm_dg_filter: NULL argument");
  if (ctx->prm.filter_order <= 0) return fail(CM_DG_ESTATE, "cm_dg_filter: the ctx was set up with filter_order = 0");
  int rc = enter(ctx, "cm_dg_filter"); if (rc) return rc;
  FilterArgs a;
  a.Nq = ctx->Nq; a.Np = ctx->Np; a.nvar = ctx->nvar; a.general = ctx->general; a.use_ref = ctx->prm.use_ref;
  a.stride = ctx->stride; a.Q = Q_dev; a.erow = ctx->d_erow; a.ztab = ctx->d_ztab; a.ref = ctx->d_ref;
  for (int i = 0; i < CM_MAXNQ; ++i) for (int j = 0; j < CM_MAXNQ; ++j) a.F[i][j] = ctx->Filt[i][j];
  {
    Timed tm(ctx, 2);
    filter_kernel<<<(unsigned)ctx->Ne, 128, 2 * ctx->Np * sizeof(double), ctx->st>>>(a);
  }
  CM_CUDA(cudaGetLastError());
  return CM_DG_OK;
}

// the launches of ONE time step on the ctx stream
static int one_step(cm_dg_ctx* ctx, double* Q_dev, double dt, int nstages, const double* A, const double* B) {
  const size_t bytes = (size_t)ctx->nvar * ctx->stride * sizeof(double);
  // A stage never updates in place (neighbours still read the old state).  The stages cycle
  // Q_dev -> Q2 -> Q3 -> Q2 -> ... -> Q_dev: the last stage of a step writes the caller's array, no copy is appended
  // (a one-stage scheme writes Q2 and is copied back).
  int rc;
  double* src = Q_dev;
  for (int st = 0; st < nstages; ++st) {
    double* dst = (st == nstages - 1 && nstages > 1) ? Q_dev : ((st & 1) ? ctx->d_Q3 : ctx->d_Q2);
    if (ctx->prm.sgs) { rc = run_gradient(ctx, src, ctx->d_G, 0); if (rc) return rc; }
    rc = run_tendency(ctx, src, ctx->d_res, dst, 1, A[st], B[st], dt);
    if (rc) return rc;
    src = dst;
  }
  if (nstages == 1) CM_CUDA(cudaMemcpyAsync(Q_dev, ctx->d_Q2, bytes, cudaMemcpyDeviceToDevice, ctx->st));
  if (ctx->prm.filter_order > 0) { rc = cm_dg_filter(ctx, Q_dev); if (rc) return rc; }
  return CM_DG_OK;
}

int cm_dg_lsrk_step_table(cm_dg_ctx* ctx, double* Q_dev, double t, double dt, int32_t nsteps, int32_t nstages,
                          const double* A, const double* B, const double* C) {
  (void)t; (void)C;   // no time-dependent forcing on this path (reading R14)
  if (!ctx || !Q_dev || !A || !B) return fail(CM_DG_EINVAL, "cm_dg_lsrk_step_table: NULL argument");
  if (nsteps < 0 || nstages < 1) return fail(CM_DG_EINVAL, "cm_dg_lsrk_step_table: nsteps must be >= 0 and nstages >= 1");
  if (A[0] != 0.0) return fail(CM_DG_EINVAL, "cm_dg_lsrk_step_table: A[0] must be 0 (the residual starts from zero)");
  int rc = enter(ctx, "cm_dg_lsrk_step_table"); if (rc) return rc;
  // CUDA graph of one step: every kernel argument (state pointers of the stage ring, dt, A_s, B_s) is fixed by
  // (Q_dev, dt, table), so the step captured for that key can be replayed.  Captured on the second consecutive call with the
  // same key (the first one has configured every kernel on this device); never while the per-launch events of
  // cm_dg_profile_begin are on; any failure (e.g. the legacy default stream cannot be captured) falls back to plain launches.
  if (ctx->graphs && !ctx->profiling && nsteps > 0) {
    cm_dg_ctx::StepKey key;
    key.Q = Q_dev; key.dt = dt; key.nstages = nstages;
    key.A.assign(A, A + nstages); key.B.assign(B, B + nstages);
    if (ctx->step_exec && key == ctx->step_key) {
      for (int s = 0; s < nsteps; ++s) CM_CUDA(cudaGraphLaunch(ctx->step_exec, ctx->st));
      return CM_DG_OK;
    }
    if (key == ctx->last_key) {
      if (ctx->step_exec) { cudaGraphExecDestroy(ctx->step_exec); ctx->step_exec = nullptr; }
      cudaGraph_t graph = nullptr;
      if (cudaStreamBeginCapture(ctx->st, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
        const int rs = one_step(ctx, Q_dev, dt, nstages, A, B);
        const cudaError_t ee = cudaStreamEndCapture(ctx->st, &graph);
        if (rs == CM_DG_OK && ee == cudaSuccess && graph && cudaGraphInstantiate(&ctx->step_exec, graph, 0) == cudaSuccess)
          ctx->step_key = key;
        else
          ctx->step_exec = nullptr;
        if (graph) cudaGraphDestroy(graph);
      }
      cudaGetLastError();                                  // a refused capture is not an error of this call
      if (ctx->step_exec) {
        for (int s = 0; s < nsteps; ++s) CM_CUDA(cudaGraphLaunch(ctx->step_exec, ctx->st));
        return CM_DG_OK;
      }
      ctx->graphs = false;                                 // do not try again on this ctx
    }
    ctx->last_key = key;
  }
  for (int s = 0; s < nsteps; ++s) { rc = one_step(ctx, Q_dev, dt, nstages, A, B); if (rc) return rc; }
  return CM_DG_OK;
}

int cm_dg_lsrk_step(cm_dg_ctx* ctx, double* Q_dev, double t, double dt, int32_t nsteps) {
  return cm_dg_lsrk_step_table(ctx, Q_dev, t, dt, nsteps, 5, kRKA, kRKB, nullptr);
}

int cm_dg_diagnostics(cm_dg_ctx* ctx, const double* Q_dev, cm_dg_diag* out) {
  if (!ctx || !Q_dev || !out) return fail(CM_DG_EINVAL, "cm_dg_diagnostics: NULL argument");
  { int rc_ = enter(ctx, "cm_dg_diagnostics"); if (rc_) return rc_; }
  DiagArgs a;
  a.Nq = ctx->Nq; a.Np = ctx->Np; a.nvar = ctx->nvar; a.general = ctx->general; a.use_ref = ctx->prm.use_ref;
  a.Ne = ctx->Ne; a.stride = ctx->stride; a.Q = Q_dev; a.geo = ctx->d_geo; a.erow = ctx->d_erow; a.ztab = ctx->d_ztab;
  a.Jflat = 1.0 / ctx->kp.invJ; for (int i = 0; i < CM_MAXNQ; ++i) a.w[i] = ctx->w[i];
  a.th = ctx->kp.th; a.satadj = ctx->kp.satadj;
  const int thr = 128;
  {
    Timed tm(ctx, 2);
    diag_kernel<<<(unsigned)ctx->Ne, thr, 7 * thr * sizeof(double), ctx->st>>>(a, ctx->d_part);
  }
  CM_CUDA(cudaGetLastError());
  double* d_red = ctx->d_lev + (size_t)ctx->prm.ne[2] * ctx->Nq * (CM_DG_NPROF + 1);
  {
    // two fixed-order stages: 256 blocks over contiguous element ranges, then one block over their results
    Timed tm(ctx, 2);
    const int nb = 256;
    const long long chunk = (ctx->Ne + nb - 1) / nb;
    diag_reduce_kernel<<<nb, 256, 0, ctx->st>>>(ctx->Ne, chunk, ctx->d_part, d_red + 8);
    diag_reduce_kernel<<<1, 256, 0, ctx->st>>>(nb, nb, d_red + 8, d_red);
  }
  CM_CUDA(cudaGetLastError());
  double s[7] = {0, 0, 0, 0, 0, 0, 0};
  CM_CUDA(cudaMemcpyAsync(s, d_red, sizeof(s), cudaMemcpyDeviceToHost, ctx->st));
  CM_CUDA(cudaStreamSynchronize(ctx->st));
  out->mass = s[0]; out->energy = s[1]; out->water = s[2]; out->kinetic = s[3] / s[4]; out->volume = s[4];
  out->max_wavespeed = s[5]; out->n_nonfinite = (int64_t)s[6]; out->min_node_dx = ctx->min_node_dx;
  return CM_DG_OK;
}

int cm_dg_profiles(cm_dg_ctx* ctx, const double* Q_dev, double* out, int32_t nlev_capacity) {
  if (!ctx || !Q_dev || !out) return fail(CM_DG_EINVAL, "cm_dg_profiles: NULL argument");
  { int rc_ = enter(ctx, "cm_dg_profiles"); if (rc_) return rc_; }
  const int nlev = ctx->prm.ne[2] * ctx->Nq;
  if (nlev_capacity < nlev) return fail(CM_DG_EINVAL, "cm_dg_profiles: out_host holds fewer than Ez * Nq levels");
  ProfArgs a;
  a.Nq = ctx->Nq; a.Np = ctx->Np; a.nvar = ctx->nvar; a.general = ctx->general;
  a.Ne = ctx->Ne; a.stride = ctx->stride; a.Q = Q_dev; a.geo = ctx->d_geo; a.erow = ctx->d_erow; a.ztab = ctx->d_ztab;
  a.lev = ctx->d_lev; a.A3flat = ctx->kp.cA[2]; a.grav = ctx->prm.grav;
  for (int i = 0; i < CM_MAXNQ; ++i) a.w[i] = ctx->w[i];
  a.th = ctx->kp.th; a.satadj = ctx->kp.satadj;
  ProfRedArgs r;
  r.Nq = ctx->Nq; r.Ex = ctx->prm.ne[0]; r.Ey = ctx->prm.ne[1]; r.Ez = ctx->prm.ne[2];
  r.L = ctx->tileL; r.PY = ctx->tilePY; r.NXC = r.Ex / r.L;
  r.flat_z = ctx->general ? 0 : 1; r.flat_lo = ctx->prm.lo[2]; r.flat_h = ctx->h[2]; r.flat_dz0 = 0.0;
  for (int i = 0; i < CM_MAXNQ; ++i) r.xi[i] = ctx->xi[i];
  double* part = ctx->d_res;                               // scratch: Ne * Nq * 12 <= Ne * Np * nvar doubles
  double* sumW = ctx->d_lev + (size_t)nlev * CM_DG_NPROF;
  const int NF = ctx->Nq * ctx->Nq;
  for (int pass = 0; pass < 2; ++pass) {
    a.pass = r.pass = pass;
    Timed tm(ctx, 2);
    prof_kernel<<<(unsigned)ctx->Ne, 64, (size_t)NF * PROF_NS1 * sizeof(double), ctx->st>>>(a, part);
    prof_reduce_kernel<<<(unsigned)nlev, 256, 0, ctx->st>>>(r, part, ctx->d_lev, sumW);
  }
  CM_CUDA(cudaGetLastError());
  CM_CUDA(cudaMemcpyAsync(out, ctx->d_lev, (size_t)nlev * CM_DG_NPROF * sizeof(double), cudaMemcpyDeviceToHost, ctx->st));
  CM_CUDA(cudaStreamSynchronize(ctx->st));
  return CM_DG_OK;
}

static int stage_buffer(cm_dg_ctx* ctx, size_t bytes) {
  if (!ctx->d_stage) CM_CUDA(cudaMalloc(&ctx->d_stage, 2 * bytes));
  return CM_DG_OK;
}

int cm_dg_rhs_host(cm_dg_ctx* ctx, const double* Q_host, double* dQ_host, double t) {
  if (!ctx || !Q_host || !dQ_host) return fail(CM_DG_EINVAL, "cm_dg_rhs_host: NULL argument");
  { int rc_ = enter(ctx, "cm_dg_rhs_host"); if (rc_) return rc_; }
  const size_t bytes = (size_t)ctx->nvar * ctx->stride * sizeof(double);
  int rc = stage_buffer(ctx, bytes); if (rc) return rc;
  double* dq = ctx->d_stage; double* dd = ctx->d_stage + (size_t)ctx->nvar * ctx->stride;
  CM_CUDA(cudaMemcpyAsync(dq, Q_host, bytes, cudaMemcpyHostToDevice, ctx->st));
  rc = cm_dg_rhs(ctx, dq, dd, t); if (rc) return rc;
  CM_CUDA(cudaMemcpyAsync(dQ_host, dd, bytes, cudaMemcpyDeviceToHost, ctx->st));
  CM_CUDA(cudaStreamSynchronize(ctx->st));
  return CM_DG_OK;
}

int cm_dg_lsrk_step_host(cm_dg_ctx* ctx, double* Q_host, double t, double dt, int32_t nsteps) {
  if (!ctx || !Q_host) return fail(CM_DG_EINVAL, "cm_dg_lsrk_step_host: NULL argument");
  { int rc_ = enter(ctx, "cm_dg_lsrk_step_host"); if (rc_) return rc_; }
  const size_t bytes = (size_t)ctx->nvar * ctx->stride * sizeof(double);
  int rc = stage_buffer(ctx, bytes); if (rc) return rc;
  double* dq = ctx->d_stage;
  CM_CUDA(cudaMemcpyAsync(dq, Q_host, bytes, cudaMemcpyHostToDevice, ctx->st));
  rc = cm_dg_lsrk_step(ctx, dq, t, dt, nsteps); if (rc) return rc;
  CM_CUDA(cudaMemcpyAsync(Q_host, dq, bytes, cudaMemcpyDeviceToHost, ctx->st));
  CM_CUDA(cudaStreamSynchronize(ctx->st));
  return CM_DG_OK;
}

int cm_dg_profile_begin(cm_dg_ctx* ctx) {
  if (!ctx) return fail(CM_DG_EINVAL, "cm_dg_profile_begin: NULL ctx");
  ctx->profiling = true; ctx->ev_used = 0;
  return CM_DG_OK;
}

int cm_dg_profile_end(cm_dg_ctx* ctx, cm_dg_kernel_stats* out) {
  if (!ctx || !out) return fail(CM_DG_EINVAL, "cm_dg_profile_end: NULL argument");
  if (!ctx->profiling) return fail(CM_DG_ESTATE, "cm_dg_profile_end: profiling was not started");
  ctx->profiling = false;
  CM_CUDA(cudaStreamSynchronize(ctx->st));
  std::memset(out, 0, sizeof(*out));
  for (size_t k = 0; k + 1 < ctx->ev_used + 1 && k < ctx->ev_used; k += 2) {
    float ms = 0.f;
    CM_CUDA(cudaEventElapsedTime(&ms, ctx->ev[k], ctx->ev[k + 1]));
    const int kind = ctx->ev_kind[k / 2];
    if (kind == 0) { out->launches_gradient++; out->ms_gradient += ms; }
    else if (kind == 1) { out->launches_tendency++; out->ms_tendency += ms; }
    else { out->launches_other++; out->ms_other += ms; }
  }
  ctx->ev_used = 0;
  return CM_DG_OK;
}

}  // extern "C"

// ------------------------------------------------------------------ a6 without a ctx: cm_dg_diagnostics_static
// For callers that may not obtain device memory (a pool that owns the whole GPU, an attached monitor without a budget, a
// loop that cannot afford cudaMalloc's device-wide synchronisation; see include/cm_dg.h): the partial sums that
// cm_dg_diagnostics keeps in ctx-owned cudaMalloc'd buffers live here in one array built into the library image.
// Layout in doubles: [0, 8) totals | [8, 8 + 7*256) block sums | then 7 per element, CM_DG_STATIC_MAX_ELEM elements.
// Every device that loads this module carries the array until the process ends.
static __device__ __align__(256) double cm_static_scratch[CM_DG_STATIC_SCRATCH_BYTES / sizeof(double)];

namespace {

struct DiagStaticArgs {
  int Nq, Np, nvar;
  long long stride;
  const double* Q; const double* J; const double* z;
  double w[CM_MAXNQ];
  double R_d, c_vd, a, b, T_0, I_v0, grav;   // a = R_v - R_d, b = c_vv - c_vd (eq. 7-8)
};

// diag_kernel with the Jacobian determinant and the height read from caller arrays (no ctx geometry, no z table):
// per-element sums {mass, energy, water, M |u|^2 / 2, M, max(|u| + c), non-finite count} into part[7 e ..].  `part` is the
// DEVICE address of cm_static_scratch as returned by cudaGetSymbolAddress, handed in by the host like any other pointer.
__global__ void diag_static_kernel(const __grid_constant__ DiagStaticArgs a, double* __restrict__ part) {
  extern __shared__ double sh[];
  const long long e = blockIdx.x;
  double s[7] = {0, 0, 0, 0, 0, 0, 0};
  for (int n = threadIdx.x; n < a.Np; n += blockDim.x) {
    const int i = n % a.Nq, j = (n / a.Nq) % a.Nq, k = n / (a.Nq * a.Nq);
    const long long idx = e * a.Np + n;
    double Y[6] = {0, 0, 0, 0, 0, 0};
    for (int v = 0; v < a.nvar; ++v) { Y[v] = a.Q[v * a.stride + idx]; if (!isfinite(Y[v])) s[6] += 1.0; }
    const double M = a.w[i] * a.w[j] * a.w[k] * a.J[idx];
    const double Phi = a.grav * a.z[idx];
    const double ir = 1.0 / Y[0];
    const double u2 = (Y[1] * Y[1] + Y[2] * Y[2] + Y[3] * Y[3]) * ir * ir;
    const double q = (a.nvar == 6) ? Y[5] * ir : 0.0;
    const double cvm = a.c_vd + a.b * q, Rm = a.R_d + a.a * q;
    const double eint = Y[4] * ir - 0.5 * u2 - Phi;
    const double T = a.T_0 + (eint - q * a.I_v0) / cvm;
    const double c = sqrt((1.0 + Rm / cvm) * Rm * T);
    s[0] += M * Y[0]; s[1] += M * Y[4]; s[2] += M * Y[5]; s[3] += M * 0.5 * u2; s[4] += M;
    s[5] = fmax(s[5], sqrt(u2) + c);
  }
  for (int m = 0; m < 7; ++m) sh[m * blockDim.x + threadIdx.x] = s[m];
  __syncthreads();
  if (threadIdx.x == 0) {
    double r[7] = {0, 0, 0, 0, 0, 0, 0};
    for (int t = 0; t < blockDim.x; ++t)
      for (int m = 0; m < 7; ++m) r[m] = (m == 5) ? fmax(r[m], sh[m * blockDim.x + t]) : r[m] + sh[m * blockDim.x + t];
    for (int m = 0; m < 7; ++m) part[7 * e + m] = r[m];
  }
}

// Device address of cm_static_scratch on the current device.  In host code the name `cm_static_scratch` is only a handle for
// the runtime's symbol table (passing it to a kernel would hand the GPU a host address), so the address is asked for once
// per device with that device current, checked, and remembered.  Devices beyond the table are looked up on every call.
constexpr int kStaticMaxDev = 64;
std::mutex g_static_mu;
double* g_static_ptr[kStaticMaxDev] = {nullptr};

int static_scratch(double** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0)
    return fail(CM_DG_ECUDA, "cm_dg_diagnostics_static: no current CUDA device (this library has no CPU path)");
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (dev < kStaticMaxDev && g_static_ptr[dev]) { *out = g_static_ptr[dev]; return CM_DG_OK; }
  double* ptr = nullptr;
  const cudaError_t err = cudaGetSymbolAddress((void**)&ptr, cm_static_scratch);
  if (err != cudaSuccess || !ptr)
    return fail(CM_DG_ECUDA, std::string("cm_dg_diagnostics_static: cudaGetSymbolAddress(cm_static_scratch) on device ") +
                             std::to_string(dev) + ": " + cudaGetErrorString(err));
  if (dev < kStaticMaxDev) g_static_ptr[dev] = ptr;
  *out = ptr;
  return CM_DG_OK;
}

}  // namespace

extern "C" int cm_dg_diagnostics_static(const cm_dg_static_desc* d, const double* Q_dev, const double* J_dev, const double* z_dev,
                                        void* cuda_stream, cm_dg_diag* out) {
  if (!d || !Q_dev || !J_dev || !z_dev || !out) return fail(CM_DG_EINVAL, "cm_dg_diagnostics_static: NULL argument");
  if (d->N < 1 || d->N > 7) return fail(CM_DG_EINVAL, "cm_dg_diagnostics_static: polynomial order N must be in 1..7");
  if (d->nvar != 5 && d->nvar != 6) return fail(CM_DG_EINVAL, "cm_dg_diagnostics_static: nvar must be 5 or 6");
  if (d->n_elem < 1) return fail(CM_DG_EINVAL, "cm_dg_diagnostics_static: n_elem must be >= 1");
  if (d->n_elem > CM_DG_STATIC_MAX_ELEM)
    return fail(CM_DG_EINVAL, "cm_dg_diagnostics_static: n_elem = " + std::to_string((long long)d->n_elem) +
                              " exceeds CM_DG_STATIC_MAX_ELEM = " + std::to_string(CM_DG_STATIC_MAX_ELEM) +
                              " (the built-in scratch array holds 7 sums per element and cannot grow; use cm_dg_diagnostics"
                              " on a ctx for larger meshes)");
  const int Nq = d->N + 1, Np = Nq * Nq * Nq;
  if (d->field_stride < d->n_elem * Np) return fail(CM_DG_EINVAL, "cm_dg_diagnostics_static: field_stride is smaller than n_elem * (N+1)^3");
  if (!(d->c_vd > 0.0) || !(d->R_d > 0.0)) return fail(CM_DG_EINVAL, "cm_dg_diagnostics_static: R_d and c_vd must be positive");
  double* scratch = nullptr;
  { int rc_ = static_scratch(&scratch); if (rc_) return rc_; }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  DiagStaticArgs a;
  a.Nq = Nq; a.Np = Np; a.nvar = d->nvar; a.stride = d->field_stride; a.Q = Q_dev; a.J = J_dev; a.z = z_dev;
  {
    double xi[CM_MAXNQ], D[CM_MAXNQ][CM_MAXNQ];
    for (int i = 0; i < CM_MAXNQ; ++i) a.w[i] = 0.0;
    lgl_operators(d->N, xi, a.w, D);
  }
  a.R_d = d->R_d; a.c_vd = d->c_vd; a.a = d->R_v - d->R_d; a.b = d->c_vv - d->c_vd; a.T_0 = d->T_0; a.I_v0 = d->I_v0; a.grav = d->grav;
  double* total = scratch; double* blk = scratch + 8; double* part = scratch + 8 + 7 * 256;
  const int thr = 128, nb = 256;
  diag_static_kernel<<<(unsigned)d->n_elem, thr, 7 * thr * sizeof(double), st>>>(a, part);
  CM_CUDA(cudaGetLastError());
  // the same two fixed-order stages as cm_dg_diagnostics; all nb block rows and all 7 totals are rewritten on every call
  const long long chunk = (d->n_elem + nb - 1) / nb;
  diag_reduce_kernel<<<nb, 256, 0, st>>>(d->n_elem, chunk, part, blk);
  diag_reduce_kernel<<<1, 256, 0, st>>>(nb, nb, blk, total);
  CM_CUDA(cudaGetLastError());
  double s[7] = {0, 0, 0, 0, 0, 0, 0};
  CM_CUDA(cudaMemcpyAsync(s, total, sizeof(s), cudaMemcpyDeviceToHost, st));
  CM_CUDA(cudaStreamSynchronize(st));
  out->mass = s[0]; out->energy = s[1]; out->water = s[2]; out->kinetic = s[3] / s[4]; out->volume = s[4];
  out->max_wavespeed = s[5]; out->n_nonfinite = (int64_t)s[6]; out->min_node_dx = 0.0;
  return CM_DG_OK;
}
