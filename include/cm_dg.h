/* cm_dg.h -- C ABI of the B200-native nodal-DG right-hand side for atmospheric LES
 * (hot path of arXiv 2110.00853, "Large-eddy simulations with ClimateMachine").
 *
 * P:L<n> below = line n of the paper text.  The library evaluates, in fp64 on one GPU,
 *
 *     dY/dt = -div(F1(Y) + F2(Y, grad Y)) + S(Y)                                  eq. (16)
 *
 * for Y = [rho, rho*u, rho*v, rho*w, rho*e_tot, (rho*q_tot)] on a structured brick of hexahedral
 * elements with (N+1)^3 Legendre-Gauss-Lobatto nodes each (eq. 17), discretised by the nodal
 * discontinuous-Galerkin method of eq. (26)/(32) with the Rusanov flux (eq. 27), the
 * BR1 auxiliary gradient (eq. 28-31), the Smagorinsky-Lilly closure (eq. 33-38),
 * reflecting free-slip walls (App. A3) and the 2N-storage LSRK54 scheme.
 *
 * Conventions
 *   - Every pointer is tagged HOST or DEVICE.  Nothing here is a torch type; the caller allocates device
 *     memory however it likes (the Python binding uses torch.empty(..., device="cuda")).
 *   - State layout (DEVICE and the *_host variants alike): structure of arrays, fp64,
 *         Q[v * field_stride + e * np + n],   v = rho, rho*u, rho*v, rho*w, rho*e_tot, [rho*q_tot]
 *     e = element in LIBRARY order (0 <= e < n_elem), n = i + Nq*(j + Nq*k) with i along x (xi) fastest,
 *     Nq = N+1, np = Nq^3.  cm_dg_layout() reports field_stride (>= n_elem*np, a multiple of 32 doubles)
 *     and lex_of_elem[e] = ex + Ex*(ey + Ey*ez), the lexicographic id of library element e (the library
 *     orders elements in small spatial tiles so that face neighbours stay close in memory / in L2).
 *   - All calls on one ctx are issued on the CUDA stream given to cm_dg_setup (0 = legacy default stream).
 *     cm_dg_rhs / cm_dg_lsrk_step / cm_dg_gradient are asynchronous and never synchronise;
 *     cm_dg_diagnostics, cm_dg_profile_end and the *_host variants synchronise that stream.
 *   - Return value: CM_DG_OK (0) or a negative code; cm_dg_last_error() gives a thread-local message.
 *     No exception or abort crosses this boundary.  Non-finite state values are reported by
 *     cm_dg_diagnostics (n_nonfinite), never trapped.
 *   - There is NO CPU fallback: without a CUDA device cm_dg_setup fails with CM_DG_ECUDA.
 */
#ifndef CM_DG_H
#define CM_DG_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CM_DG_OK 0
#define CM_DG_EINVAL (-1) /* bad N / ne / nvar / NULL pointer / non-positive Jacobian / metric identity > 1e-10 */
#define CM_DG_ENOMEM (-2)
#define CM_DG_ECUDA (-3)  /* message carries cudaGetErrorString                                            */
#define CM_DG_ESTATE (-4) /* call not valid for this ctx (e.g. profile_end without profile_begin)          */

typedef struct cm_dg_ctx cm_dg_ctx; /* opaque, library-owned */

/* Problem description (all HOST memory, copied before cm_dg_setup returns). */
typedef struct {
  int32_t N;                /* polynomial order, 2..7 (the paper's runs and BASELINE use 4; the
                               sweep 3..6).  N = 1 is refused with CM_DG_EINVAL: with two LGL nodes per direction every node
                               lies on three faces, the drag law's "first layer of interior nodes" (A2) does not exist, and
                               the kernels' split into volume lines and face nodes has no interior left to overlap with;
                               no configuration of the paper or of BASELINE uses it                              */
  int32_t ne[3];            /* Ex, Ey, Ez: structured hexahedral brick                             */
  double lo[3], hi[3];      /* domain box before warping [m]                                                */
  int32_t bc[3];            /* per direction: 0 periodic, 1 impenetrable free-slip no-flux wall at both ends */
  int32_t nvar;             /* 5 dry | 6 with rho*q_tot                                                     */
  int32_t geom;             /* 0 flat brick | 1 linear-decay terrain warp of z by zsfc_nodes | 2 xyz */
  const double* zsfc_nodes; /* geom==1: HOST [Ey*Nq][Ex*Nq] surface height at the bottom nodes              */
  const double* xyz;        /* geom==2: HOST [3][Ne][Np], LEXICOGRAPHIC element order                       */
  double R_d, c_vd, R_v, c_vv, T_0, I_v0, grav; /* Table 1, eq. (9); Phi = grav * z     */
  int32_t sgs;              /* 0 inviscid | 1 Smagorinsky-Lilly (eq. 38) | 2 Vreman (eq. 39a-d)   */
  double C_s, Pr_t;         /* Smagorinsky coefficient, turbulent Prandtl number (eq. 36)                   */
  int32_t use_ref;          /* 1: remove the hydrostatic reference state in the momentum equation (eq. 4)   */
  const double *ref_rho, *ref_rhoe, *ref_rhoq; /* HOST [Ne][Np] LEXICOGRAPHIC; resting reference state;
                                                  p_r is derived from them with the library's EOS          */
  double shf_bottom;        /* W m^-2 prescribed upward energy flux through the z-low wall, 0 = none */
  /* ---- optional physics and numerics beyond the five BASELINE configs; all-zero = off / defaults ---- */
  int32_t richardson;       /* 1: multiply nu_t by the stability factor f_b of eq. (40); needs sgs != 0 */
  double p_0;               /* reference pressure of theta_v in eq. (40) [Pa]; 0 = 1e5                       */
  double sponge_alpha;      /* Rayleigh sponge (A4)-(A5): relaxation coefficient [1/s], 0 = no sponge */
  double sponge_zs;         /* height where the absorbing layer starts [m]; it ends at hi[2]                  */
  int32_t sponge_gamma;     /* power of the sine profile (positive, typically 2); 0 = 2                       */
  double u_relax[3];        /* velocity the momentum is relaxed to inside the layer [m/s]                     */
  int32_t filter_order;     /* exponential element filter of eq. (52): order s (even, e.g. 64), 0 = off;
                               when on, cm_dg_lsrk_step* apply it after every time step (cm_dg_filter applies it once) */
  double filter_alpha;      /* alpha = -log(eps_M) of eq. (52); 0 = 36.0436533891172 (double precision)       */
  int32_t riemann;          /* numerical flux of F1: 0 Rusanov (eq. 27) | 1 HLLC | 2 Roe (both named at P:L256); HLLC and
                               Roe run on the stored-metric kernels                                           */
  int32_t metric_form;      /* 0 cross-product metric terms (extruded / 2.5-D warps) | 1 curl-invariant form
                               (fully 3-D warps; geom == 2)                                                   */
  /* ---- surface fluxes through the z-low wall (App. A1; need bc[2] == 1); all-zero = free slip, no flux ---- */
  double drag_cd;           /* C_d of the aerodynamic drag law, eq. (A2): n.(rho tau) = -rho C_d |u_p,int| u_p,int
                               with u_p,int the wall-parallel velocity at the first layer of interior nodes          */
  double lhf_bottom;        /* W m^-2 latent heat flux, added to shf_bottom in the wall energy flux   */
  double evap_bottom;       /* kg m^-2 s^-1 evaporation E = n.(rho d_qv)|sfc into the domain: enters the
                               rho*q_tot and rho equations; CM_DG_EINVAL unless nvar == 6; the caller derives it from LHF */
  /* ---- equilibrium moist thermodynamics (section 2.7, eq. 15); nvar == 6; runs on the stored-metric kernels ---- */
  int32_t satadj;           /* 1: temperature and liquid water from the saturation adjustment: the root T of
                               I*(T; rho, q_tot) = I by Newton iterations, the saturation excess q_tot - q_v*(T, rho) as liquid
                               (warm phase), q_v* from the closed-form saturation vapour pressure of a calorically perfect gas
                               (Romps 2008); R_m, c_vm, p and the sound speed then include the condensate (eq. 7-8, 13-14)   */
  double c_vl;              /* isochoric heat capacity of liquid water (Table 1); 0 = 4181 J/(kg K)              */
  double p_triple, T_triple;/* triple point of water anchoring p*(T); 0 = 611.657 Pa, 273.16 K                               */
} cm_dg_params;

/* Optional scheduling knobs (HOST, copied by cm_dg_setup_tuned).  They never change what is computed (the parity tests
 * run every setting against the CPU reference of tests/), only how the work is laid out on the GPU.  All-zero = the defaults, except
 * ahead_t / ahead_g whose default is -1. */
typedef struct {
  int32_t order_lex;     /* 1: lexicographic element order instead of the tiled one (lex_of_elem becomes the identity)   */
  int32_t max_chunk;     /* tiled order: longest x-chunk L (L divides Ex), 0 = 32                                       */
  int32_t max_patch;     /* tiled order: tallest y-patch PY (PY divides Ey), 0 = 16                                     */
  int32_t force_general; /* 1: use the stored-metric kernels (the path of warped meshes) on a flat mesh too             */
  int32_t kernel;        /* 0 default | 10 row-sweep kernels (flat) | 7 CTA-per-element kernels (flat) | 11 CTA-per-element
                            tendency kernel of stored-metric meshes (their default) | 2 thread-per-node stored-metric kernels */
  int32_t ahead_t;       /* kernel 7: L2 prefetch distance of the tendency kernel in elements; -1 one wave, 0 off       */
  int32_t ahead_g;       /* same for the gradient kernel                                                                */
  int32_t row_len;       /* kernel 10: elements per row sweep (must divide the x-chunk), 0 = chosen by the library: the
                            whole chunk on large meshes, shorter rows (>= 8) where that leaves fewer than 4 waves of CTAs   */
  int32_t no_graph;      /* 1: cm_dg_lsrk_step* always launch kernel by kernel; 0: a time step is captured as a CUDA graph on
                            the second consecutive call with the same (Q_dev, dt, table) and replayed afterwards           */
  int32_t no_terrain;    /* 1: a terrain-following mesh (geom == 1) is treated like any stored-metric mesh (nine metric tiles
                            per element instead of the three that such a mesh needs)                                       */
} cm_dg_tuning;

/* Conservation integrals and step-size ingredients (eq. 57; eq. 61-62). */
typedef struct {
  double mass;          /* sum M rho,        M = w_i w_j w_k |J|                                           */
  double energy;        /* sum M rho e_tot                                                                  */
  double water;         /* sum M rho q_tot (0 when nvar == 5)                                               */
  double kinetic;       /* E_k = (1/2) sum M |u|^2 / sum M                                                  */
  double max_wavespeed; /* max over nodes of |u| + c                                                        */
  double min_node_dx;   /* smallest distance between adjacent LGL nodes of the mesh                         */
  double volume;        /* sum M                                                                            */
  int64_t n_nonfinite;  /* number of state values that are NaN or +-Inf                                     */
} cm_dg_diag;

/* Per-kernel device timings gathered between cm_dg_profile_begin and cm_dg_profile_end (CUDA events
 * recorded on the ctx stream around every launch). */
typedef struct {
  int64_t launches_gradient, launches_tendency, launches_other;
  double ms_gradient, ms_tendency, ms_other;
} cm_dg_kernel_stats;

/* a0: mesh, LGL nodes/weights, derivative matrix, metric terms (eq. 24), connectivity,
 * reference state.  `cuda_stream` is a cudaStream_t (NULL = default stream).  On success *out owns all
 * device scratch (geometry, gradient array, LSRK residual, two more state buffers); the one exception is the staging
 * buffer of the *_host calls, see there. */
int cm_dg_setup(const cm_dg_params* p, void* cuda_stream, cm_dg_ctx** out);

/* Same with explicit scheduling knobs (tuning == NULL: defaults).  CM_DG_EINVAL for an unknown kernel id or a row_len
 * that does not divide the x-chunk.  After any refusal *out is NULL. */
int cm_dg_setup_tuned(const cm_dg_params* p, const cm_dg_tuning* tuning, void* cuda_stream, cm_dg_ctx** out);

/* Layout of state arrays: n_elem, np, field_stride (doubles) and, if non-NULL, lex_of_elem (HOST, n_elem
 * int32 entries).  Any output pointer may be NULL. */
int cm_dg_layout(const cm_dg_ctx* ctx, int64_t* n_elem, int32_t* np, int64_t* field_stride, int32_t* lex_of_elem);

/* Nodal coordinates in library layout: xyz_dev is DEVICE [3][field_stride]. */
int cm_dg_coords(cm_dg_ctx* ctx, double* xyz_dev);

/* Metric terms as used by the kernels (tests): Ja_dev DEVICE [9][field_stride] with Ja[3*d+c] = J dxi_d/dx_c
 * (cross-product form), J_dev DEVICE [field_stride] = det(dx/dxi). */
int cm_dg_metrics(cm_dg_ctx* ctx, double* Ja_dev, double* J_dev);

/* a2: BR1 auxiliary gradient (eq. 28-31): G_dev DEVICE [15][field_stride], G[3*s+c] = d s/d x_c for
 * s = u, v, w, h_tot, q_tot (q rows are zero when nvar == 5).  Diagnostic entry point: cm_dg_rhs and
 * cm_dg_lsrk_step run the same kernel but keep its output in a packed internal form. */
int cm_dg_gradient(cm_dg_ctx* ctx, const double* Q_dev, double* G_dev);

/* a1-a4: dQ := RHS(Q, t) of eq. (32).  Q_dev, dQ_dev DEVICE [nvar][field_stride], distinct buffers. */
int cm_dg_rhs(cm_dg_ctx* ctx, const double* Q_dev, double* dQ_dev, double t);

/* a1-a5: advance Q by nsteps LSRK54 steps of size dt; every stage is one gradient kernel plus one fused
 * tendency + low-storage update kernel (replayed from a CUDA graph of one step once the same Q_dev, dt have been seen twice).  The result is left in Q_dev: the five stages of a step cycle through two
 * ctx-owned buffers and end in the caller's array (no stage updates in place, no copy is appended). */
int cm_dg_lsrk_step(cm_dg_ctx* ctx, double* Q_dev, double t, double dt, int32_t nsteps);

/* The same for any 2N-storage Runge-Kutta scheme given by its coefficient tables (HOST, nstages entries each; A[0]
 * must be 0): for s: dU <- A_s dU + dt RHS(U, t + C_s dt); U <- U + B_s dU.  cm_dg_lsrk_step is this call
 * with the Carpenter-Kennedy (5,4) table; the 14-stage scheme the paper ran is a table of 14.  C may be NULL
 * (no time-dependent forcing on this path).  CM_DG_EINVAL for nstages < 1 or A[0] != 0. */
int cm_dg_lsrk_step_table(cm_dg_ctx* ctx, double* Q_dev, double t, double dt, int32_t nsteps, int32_t nstages,
                          const double* A, const double* B, const double* C);

/* Exponential element filter of eq. (52) applied once, in place: Q <- Q_ref + (F x F x F)(Q - Q_ref) on every element and
 * prognostic field, F = V diag(exp(-alpha (n/N)^s)) V^-1 in the Legendre basis.  CM_DG_ESTATE if filter_order == 0. */
int cm_dg_filter(cm_dg_ctx* ctx, double* Q_dev);

/* a6: conservation integrals etc. of Q_dev into *out_host; synchronises the stream. */
int cm_dg_diagnostics(cm_dg_ctx* ctx, const double* Q_dev, cm_dg_diag* out_host);

/* a6 without a ctx and without any device allocation.
 *
 * Who this is for: code that holds a state array on the GPU but is not in a position to obtain device memory through
 * the CUDA allocator, and therefore cannot call cm_dg_setup (which cudaMallocs geometry, gradient and stage buffers).
 * Typical cases: (1) a host application whose memory pool (a framework's caching allocator, an RMM-style arena) has
 * already claimed the whole device, so a raw cudaMalloc beside it fails or eats into the pool's head-room; (2) a
 * monitoring tool attached to a running model (for instance through CUDA IPC handles, or under an MPS memory limit) with
 * no memory budget of its own; (3) a time loop that must not stall, because cudaMalloc and cudaFree synchronise the whole
 * device.  For them the per-element partial sums of the conservation integrals live in ONE array that is compiled into
 * the library (`static __device__`, CM_DG_STATIC_SCRATCH_BYTES = 3 684 416 bytes).  Every GPU on which the library's
 * device code gets loaded holds that array until the process exits, whether or not this function is ever called.
 *
 * What it computes: the same sums as cm_dg_diagnostics (eq. 57; eq. 61-62) with the dry / unsaturated
 * equation of state (eq. 6-10; no saturation adjustment), from arrays the caller provides in the library's layout:
 *   Q_dev  DEVICE [nvar][field_stride]   state
 *   J_dev  DEVICE [n_elem * np]          det(dx/dxi) per node (what cm_dg_metrics writes to J_dev)
 *   z_dev  DEVICE [n_elem * np]          height of every node [m], Phi = grav * z (row 2 of what cm_dg_coords writes)
 * The element order is irrelevant to these sums.  out_host (HOST) receives the result; min_node_dx is set to 0 (this call
 * does not know the mesh).  `cuda_stream` is a cudaStream_t (NULL = default stream); the call synchronises it.
 *
 * Limits and rules:
 *   - n_elem <= CM_DG_STATIC_MAX_ELEM; a larger mesh is refused with CM_DG_EINVAL and a message that names the limit
 *     (nothing is launched).  N in 1..7, nvar 5 or 6, field_stride >= n_elem * (N+1)^3.
 *   - It never calls cudaMalloc, cudaFree or any allocating library routine; the only device memory it writes is the
 *     built-in array.  The result reaches the host by one 56-byte cudaMemcpyAsync.
 *   - The first call on each device (with that device current) looks up the device address of the built-in array
 *     (cudaGetSymbolAddress) and remembers it; later calls on that device reuse it.  Make that first call before any
 *     stream capture is started on the device.
 *   - All calls on one device share the array, and it keeps whatever the previous call left there.  Nothing in it has
 *     to start at zero: every entry a call reads (n_elem x 7 partial sums, 256 x 7 block sums, 7 totals) is written
 *     earlier in the same call, so a smaller mesh after a larger one never sees stale sums.  Two calls that overlap on
 *     the same GPU (two streams, two host threads, two ctx-free users in one process) race on it: serialise them. */
#define CM_DG_STATIC_MAX_ELEM 65536
#define CM_DG_STATIC_SCRATCH_BYTES ((8 + 7 * 256 + 7 * CM_DG_STATIC_MAX_ELEM) * 8)
typedef struct {
  int32_t N;                 /* polynomial order, 1..7                                                      */
  int32_t nvar;              /* 5 dry | 6 with rho*q_tot                                                    */
  int64_t n_elem;            /* elements in Q_dev, 1..CM_DG_STATIC_MAX_ELEM                                 */
  int64_t field_stride;      /* doubles between consecutive fields of Q_dev                                 */
  double R_d, c_vd, R_v, c_vv, T_0, I_v0, grav; /* as in cm_dg_params                                       */
} cm_dg_static_desc;
int cm_dg_diagnostics_static(const cm_dg_static_desc* desc, const double* Q_dev, const double* J_dev, const double* z_dev,
                             void* cuda_stream, cm_dg_diag* out_host);

/* Density-weighted horizontal statistics of App. B (eq. B1-B4) on the nodal mesh.  Levels are the nodal
 * zeta-planes of every element layer, l = ez * Nq + k (nlev = Ez * Nq; the two planes of an element interface are separate
 * levels); <a>_l = sum W a / sum W over the plane with W = w_i w_j |Ja^3| (area element of the zeta = const surface).
 * out_host is HOST [nlev][CM_DG_NPROF], columns: <z>, <rho>, then for phi = u, v, w, h_tot, q_tot, theta_v the Favre mean
 * phibar = <rho phi>/<rho> (B1), the vertical eddy flux <rho w' phi'>/<rho> (B2) and the variance <rho phi'^2>/<rho> (B4),
 * phi' = phi - phibar (B3): 2 + 3 * 6 columns.  Two sweeps over Q_dev (means, then fluctuations), summed in a fixed order
 * (bitwise repeatable).  Uses the LSRK residual buffer as scratch; synchronises the stream.
 * CM_DG_EINVAL if nlev_capacity < Ez * Nq. */
#define CM_DG_NPROF 20
int cm_dg_profiles(cm_dg_ctx* ctx, const double* Q_dev, double* out_host, int32_t nlev_capacity);

/* End-to-end variants on HOST buffers in the same [nvar][field_stride] layout (pinned memory recommended):
 * host->device copy, the device call above, device->host copy, stream synchronise.  The device staging buffer
 * (2 x nvar x field_stride doubles) is NOT part of what cm_dg_setup allocates: the first *_host call on a ctx cudaMallocs it
 * (CM_DG_ENOMEM if that fails) and cm_dg_destroy frees it, so a ctx that is only ever driven with device pointers does not
 * pay for it.  Make that first call outside any stream capture and outside a timed region. */
int cm_dg_rhs_host(cm_dg_ctx* ctx, const double* Q_host, double* dQ_host, double t);
int cm_dg_lsrk_step_host(cm_dg_ctx* ctx, double* Q_host, double t, double dt, int32_t nsteps);

/* Kernel timing (measurement support). */
int cm_dg_profile_begin(cm_dg_ctx* ctx);
int cm_dg_profile_end(cm_dg_ctx* ctx, cm_dg_kernel_stats* out_host);

void cm_dg_destroy(cm_dg_ctx* ctx);
const char* cm_dg_last_error(void); /* thread-local, never NULL */

#ifdef __cplusplus
}
#endif
#endif /* CM_DG_H */
