"""Pins for the oracle functions of the NEXT rows of the scope table: Vreman eddy viscosity and the Richardson factor
(eq. 39-40), Rayleigh sponge (A4-A5), exponential element filter (eq. 52), 2N-storage
Runge-Kutta with any coefficient table, the HLLC flux and curl-invariant metric terms.  Every
expected value comes from the mathematics: closed forms, invariants, eigen-relations, exactness on special cases."""
import numpy as np
import pytest

import workloads as W

CS = 0.21


def _cfg(**kw):
    c = W.base_params(N=4, ne=(2, 2, 2), hi=(100.0, 200.0, 50.0), bc=(0, 0, 0), sgs=2, grav=9.81)
    c.update(kw)
    return c


def _vreman_numpy(G, Delta, Cs):
    """nu_t from the invariants of beta = alpha diag(Delta^2) alpha^T: B = ((tr beta)^2 - tr(beta^2)) / 2 (second invariant)."""
    beta = G @ np.diag(Delta ** 2) @ G.T
    B = 0.5 * (np.trace(beta) ** 2 - np.trace(beta @ beta))
    aa = np.sum(G * G)
    return 2.5 * Cs ** 2 * np.sqrt(max(B, 0.0) / aa) if aa > 0 else 0.0


# ------------------------------------------------------------------ O11: Vreman (eq. 39)
def test_vreman_vanishes_for_pure_shear_and_rank_one_gradients(oracle_mod):
    o = oracle_mod.Oracle(_cfg())
    Y = np.array([1.2, 0.0, 0.0, 0.0, 2.5e5])
    dxd = np.array([25.0, 50.0, 12.5])                  # half element sizes: Delta_m = 2 dxd / N
    G = np.zeros((6, 3)); G[0, 2] = 0.3                 # u = (alpha z, 0, 0)
    assert o.flux2(Y, G, 1.0, dxd=dxd)[1] == 0.0
    a, b = np.array([0.3, -1.0, 2.0]), np.array([0.5, 0.25, -0.125])
    G[:3] = np.outer(a, b)                              # rank one: the second invariant of beta vanishes
    assert o.flux2(Y, G, 1.0, dxd=dxd)[1] <= 1e-9 * _vreman_numpy(np.eye(3), 2 * dxd / 4, CS)
    assert o.flux2(Y, np.zeros((6, 3)), 1.0, dxd=dxd)[1] == 0.0      # no flow: 0/0 := 0


def test_vreman_closed_forms(oracle_mod):
    o = oracle_mod.Oracle(_cfg())
    Y = np.array([1.2, 0.0, 0.0, 0.0, 2.5e5])
    dxd = np.array([25.0, 50.0, 12.5]); Delta = 2 * dxd / 4
    # rotation about z: alpha = [[0, -W], [W, 0]]: beta = W^2 diag(D2^2, D1^2), B = W^4 D1^2 D2^2, alpha:alpha = 2 W^2
    Wr = 0.7
    G = np.zeros((6, 3)); G[0, 1] = -Wr; G[1, 0] = Wr
    nu = o.flux2(Y, G, 1.0, dxd=dxd)[1]
    assert abs(nu - 2.5 * CS ** 2 * Wr * Delta[0] * Delta[1] / np.sqrt(2.0)) <= 1e-14 * nu
    rng = np.random.default_rng(7)
    for _ in range(20):
        G[:3] = rng.normal(0, 1, (3, 3))
        nu = o.flux2(Y, G, 1.0, dxd=dxd)[1]
        assert abs(nu - _vreman_numpy(G[:3], Delta, CS)) <= 1e-12 * nu
    # isotropic mixing length, pure strain diag(a, -a, 0): beta = D^2 a^2 diag(1, 1, 0), B = D^4 a^4, alpha:alpha = 2 a^2
    dxd = np.array([20.0, 20.0, 20.0]); a = 0.4
    G[:3] = np.diag([a, -a, 0.0])
    nu = o.flux2(Y, G, 1.0, dxd=dxd)[1]
    assert abs(nu - 2.5 * CS ** 2 * 10.0 ** 2 * a / np.sqrt(2.0)) <= 1e-14 * nu


# ------------------------------------------------------------------ O11: Richardson factor (eq. 40)
def test_theta_v_and_richardson_factor(oracle_mod):
    cfg = _cfg(sgs=1, richardson=1, nvar=6, hi=(100.0, 100.0, 100.0))
    o = oracle_mod.Oracle(cfg)
    rho, T, q = 1.1, 285.0, 0.012
    Y = W.conserved(cfg, np.array(rho), np.array(0.0), np.array(0.0), np.array(0.0), np.array(T), np.array(q), np.array(0.0))
    P = o.primitives(Y)
    Rm = cfg["R_d"] * (1 - q) + cfg["R_v"] * q
    p = rho * Rm * T
    thv = T * (Rm / cfg["R_d"]) * (1.0e5 / p) ** (cfg["R_d"] / (cfg["c_vd"] + cfg["R_d"]))
    assert abs(P["theta_v"] - thv) <= 1e-13 * thv
    alpha = 0.02                                        # u = (alpha z, 0, 0): |S|^2 = 2 S:S = alpha^2
    J = 25.0 ** 3; Delta = 2 * 25.0 / 4
    nu_sl = (CS * Delta) ** 2 * alpha
    Pr = cfg["Pr_t"]
    for Ri, fb in ((0.0, 1.0), (-3.0, 1.0), (0.5 * Pr, 0.5 ** 0.25), (0.999 * Pr, 0.001 ** 0.25), (Pr, 0.0), (5.0, 0.0)):
        G = np.zeros((6, 3)); G[0, 2] = alpha
        G[5, 2] = Ri * alpha ** 2 * thv / cfg["grav"]   # (g / theta_v) d theta_v / dz = Ri |S|^2
        nu = o.flux2(Y, G, J)[1]
        assert abs(nu - nu_sl * fb) <= 1e-12 * nu_sl, (Ri, nu, nu_sl * fb)
    G = np.zeros((6, 3)); G[5, 2] = 1e-3                # stable, no shear: Ri = inf, f_b = 0, no NaN
    assert o.flux2(Y, G, J)[1] == 0.0


def test_theta_v_gradient_on_the_mesh_and_conservation(oracle_mod):
    cfg = W.base_params(N=4, ne=(3, 2, 3), hi=(300.0, 200.0, 600.0), bc=(0, 0, 1), sgs=2, richardson=1, nvar=6)
    o = oracle_mod.Oracle(cfg)
    xyz = o.coords(); z = xyz[..., 2]
    th0, gam, qv = 295.0, 4e-3, 0.01
    Rm = cfg["R_d"] * (1 - qv) + cfg["R_v"] * qv
    p = 1.0e5 * np.exp(-z / 8000.0)
    T = (th0 + gam * z) * (cfg["R_d"] / Rm) * (p / 1.0e5) ** (cfg["R_d"] / (cfg["c_vd"] + cfg["R_d"]))
    rho = p / (Rm * T)
    Q = W.conserved(cfg, rho, 0.01 * z, 0 * z, 0 * z, T, qv + 0 * z, z)
    G = o.gradient6(Q)
    assert np.max(np.abs(G[..., 5, 2] - gam)) <= 1e-9 * gam * 100   # nodal theta_v is linear in z up to round-off
    assert np.max(np.abs(G[..., 5, 0:2])) <= 1e-9
    # conservation of mass, energy, water with the Vreman closure and f_b on (periodic x, y; no-flux z), random state
    rng = np.random.default_rng(11)
    shp = z.shape
    Q = W.conserved(cfg, rho * (1 + 1e-3 * rng.uniform(-1, 1, shp)), *(rng.normal(0, 1.0, shp) for _ in range(3)),
                    T + 0.1 * rng.normal(0, 1, shp), qv * (1 + 0.01 * rng.uniform(-1, 1, shp)), z)
    dQ = o.rhs(Q); M = o.mass()
    for v in (0, 4, 5):
        assert abs(np.sum(M * dQ[..., v])) <= 1e-12 * np.sum(M * np.abs(dQ[..., v])), v


# ------------------------------------------------------------------ O12: Rayleigh sponge (A4-A5, R18)
def test_sponge_source_closed_form(oracle_mod):
    cfg, Q, dt = W.config4(ne=(6, 1, 5), N=3)
    zs, alpha, urel = 0.6 * cfg["hi"][2], 0.5, (10.0, 0.0, 0.0)
    cfg_s = dict(cfg); cfg_s.update(sponge_alpha=alpha, sponge_zs=zs, sponge_gamma=2, u_relax=urel)
    o0, o1 = oracle_mod.Oracle(cfg), oracle_mod.Oracle(cfg_s)
    rng = np.random.default_rng(3)
    Q = Q.copy(); Q[..., 1:4] += rng.normal(0, 1.0, Q[..., 1:4].shape)
    d = o1.rhs(Q) - o0.rhs(Q)
    z = o0.coords()[..., 2]
    tau = np.where(z > zs, alpha * np.sin(0.5 * np.pi * (z - zs) / (cfg["hi"][2] - zs)) ** 2, 0.0)
    for i in range(3):
        expect = -tau * (Q[..., 1 + i] - Q[..., 0] * urel[i])
        assert np.max(np.abs(d[..., 1 + i] - expect)) <= 1e-12 * np.max(np.abs(expect)), i
    assert np.max(np.abs(d[..., 0])) == 0.0 and np.max(np.abs(d[..., 4])) == 0.0     # momentum only (A4)
    assert np.all(d[z <= zs] == 0.0)
    assert abs(tau.max() - alpha) <= 1e-12            # tau_s(z_top) = alpha: the pi of reading R18


# ------------------------------------------------------------------ O12: exponential filter (eq. 52)
def test_filter_matrix_eigen_relations(oracle_mod):
    from numpy.polynomial import legendre as L
    for N, order in ((4, 64), (5, 8), (3, 2)):
        xi, w = oracle_mod.lgl(N)
        alpha = -np.log(2.0 ** -52)
        F = oracle_mod.filter_matrix(N, order, alpha)
        for n in range(N + 1):
            cvec = np.zeros(N + 1); cvec[n] = 1.0
            Pn = L.legval(xi, cvec)
            sigma = np.exp(-alpha * (n / N) ** order)
            assert np.max(np.abs(F @ Pn - sigma * Pn)) <= 1e-13, (N, order, n)
        assert np.max(np.abs(F.sum(axis=1) - 1.0)) <= 1e-13            # constants are kept
        assert np.max(np.abs(w @ F - w)) <= 1e-13                      # the element mean is kept (mode 0 only carries it)
        assert np.max(np.abs(F @ L.legval(xi, np.eye(N + 1)[N]))) <= 1e-15 * 10   # the top mode is removed to eps_M


def test_filter_on_the_mesh(oracle_mod):
    cfg, Q, dt = W.config5(ne=(3, 2, 3), N=4, hi=(187.5, 125.0, 3000.0))
    cfg = dict(cfg); cfg.update(filter_order=64)
    o = oracle_mod.Oracle(cfg)
    Qr = np.zeros_like(Q); Qr[..., 0] = cfg["ref_rho"]; Qr[..., 4] = cfg["ref_rhoe"]; Qr[..., 5] = cfg["ref_rhoq"]
    assert np.array_equal(o.filter(Qr), Qr)                              # the balanced background is left alone, bit for bit
    Qf = o.filter(Q)
    M = o.mass()
    for v in range(6):
        assert abs(np.sum(M * (Qf[..., v] - Q[..., v]))) <= 1e-13 * np.sum(M * np.abs(Q[..., v])), v   # conservative
    # tensor-product top mode on one element is annihilated; a trilinear perturbation passes unchanged
    from numpy.polynomial import legendre as L
    xi, _ = oracle_mod.lgl(4)
    P4 = L.legval(xi, np.eye(5)[4])
    mode = (P4[None, None, :] * P4[None, :, None] * P4[:, None, None]).reshape(-1)
    lin = ((1 + 0.3 * xi)[None, None, :] * (1 - 0.2 * xi)[None, :, None] * (1 + 0.1 * xi)[:, None, None]).reshape(-1)
    Q2 = Qr.copy(); Q2[0, :, 1] += mode; Q2[1, :, 2] += lin
    Qf = o.filter(Q2)
    assert np.max(np.abs(Qf[0, :, 1])) <= 1e-14
    assert np.max(np.abs(Qf[1, :, 2] - lin)) <= 36.05 * (1 / 4) ** 64 + 1e-14


# ------------------------------------------------------------------ O13: any 2N-storage table
def test_lsrk_table(oracle_mod):
    cfg, Q, dt = W.config1(ne=(2, 2, 2), N=3)
    o = oracle_mod.Oracle(cfg)
    A, B, Cc = oracle_mod.lsrk54_coeffs()
    assert np.array_equal(o.lsrk_table(Q, dt, 3, A, B), o.lsrk54(Q, dt, 3))
    assert np.array_equal(o.lsrk_table(Q, dt, 4, [0.0], [1.0]), o.euler(Q, dt, 4))
    # Williamson's three-stage third-order scheme: the error against a fine reference falls by ~8 per halving of dt
    A3, B3 = [0.0, -5.0 / 9.0, -153.0 / 128.0], [1.0 / 3.0, 15.0 / 16.0, 8.0 / 15.0]
    cfg, Q, _ = W.config1(ne=(2, 2, 2), N=2)
    xyz = W.node_coords(cfg); x = xyz[..., 0]
    Q = W.conserved(cfg, 1.0 + 0.2 * np.sin(2 * np.pi * x / cfg["hi"][0]), 30.0 + 0 * x, 0 * x, 0 * x, 300.0 + 0 * x, 0 * x, 0 * x)
    o = oracle_mod.Oracle(cfg)
    Tend = 0.4
    ref = o.lsrk54(Q, Tend / 256, 256)
    e = [np.max(np.abs(o.lsrk_table(Q, Tend / n, n, A3, B3) - ref)) for n in (8, 16, 32)]
    assert 6.5 < e[0] / e[1] < 9.5 and 6.5 < e[1] / e[2] < 9.5, e


# ------------------------------------------------------------------ O13: HLLC
def _state(cfg, rho, u, T, q=0.0, z=0.0):
    a = np.array
    return W.conserved(cfg, a(rho), a(u[0]), a(u[1]), a(u[2]), a(T), a(q), a(z))


def test_hllc_consistency_symmetry_contact_and_upwinding(oracle_mod):
    cfg = _cfg(sgs=0, riemann=1, nvar=6, grav=0.0)
    o = oracle_mod.Oracle(cfg)
    orus = oracle_mod.Oracle(dict(cfg, riemann=0))
    rng = np.random.default_rng(5)
    for _ in range(10):
        n = rng.normal(0, 1, 3); n /= np.linalg.norm(n)
        Ym = _state(cfg, 1.1 + 0.1 * rng.uniform(), rng.normal(0, 30, 3), 290 + 10 * rng.uniform(), 0.01)
        Yp = _state(cfg, 1.0 + 0.1 * rng.uniform(), rng.normal(0, 30, 3), 285 + 10 * rng.uniform(), 0.012)
        nF = o.flux1(Ym) @ n
        assert np.max(np.abs(o.rusanov(Ym, Ym, n) - nF)) <= 1e-12 * np.max(np.abs(nF))          # consistency
        a, b = o.rusanov(Ym, Yp, n), o.rusanov(Yp, Ym, -n)
        assert np.max(np.abs(a + b)) <= 1e-12 * np.max(np.abs(a))                               # conservation
    # isolated stationary contact: u = 0, equal pressure, density jump: HLLC keeps it (zero mass, energy, water flux,
    # pressure only in the momentum flux); Rusanov diffuses it
    n = np.array([0.0, 0.0, 1.0])
    p = 9.0e4
    Rm = cfg["R_d"] * (1 - 0.01) + cfg["R_v"] * 0.01
    YL = _state(cfg, 1.2, (0, 0, 0), p / (1.2 * Rm), 0.01); YR = _state(cfg, 0.9, (0, 0, 0), p / (0.9 * Rm), 0.01)
    F = o.rusanov(YL, YR, n)
    # (the two pressures agree to one ulp of 9e4 Pa only, so |S*| <= ulp(p) / (rho c) ~ 4e-14 m/s: fluxes of that size remain)
    assert abs(F[0]) <= 4e-14 * 1.2 and abs(F[4]) <= 4e-14 * 3.5e5 and abs(F[5]) <= 4e-14 * 0.012
    assert abs(F[3] - p) <= 1e-12 * p and abs(F[1]) + abs(F[2]) == 0.0
    assert abs(orus.rusanov(YL, YR, n)[0]) > 10.0
    # supersonic to the right: pure upwind flux of the left state
    YL = _state(cfg, 1.2, (0, 0, 900.0), 280.0, 0.01); YR = _state(cfg, 1.0, (0, 0, 850.0), 300.0, 0.01)
    assert np.array_equal(o.rusanov(YL, YR, n), o.flux1(YL) @ n)


def test_hllc_on_the_mesh_conserves_and_keeps_walls_closed(oracle_mod):
    cfg, Q, dt = W.config3(ne=(3, 2, 3), N=3, hi=(600.0, 400.0, 562.5))
    cfg = dict(cfg, riemann=1, shf_bottom=0.0)
    o = oracle_mod.Oracle(cfg)
    rng = np.random.default_rng(9)
    Q = Q.copy(); Q[..., 1:4] += rng.normal(0, 0.5, Q[..., 1:4].shape)
    dQ = o.rhs(Q); M = o.mass()
    for v in (0, 4):
        assert abs(np.sum(M * dQ[..., v])) <= 1e-12 * np.sum(M * np.abs(dQ[..., v])), v
    ds = o.rhs(Q, form="strong")
    assert np.max(np.abs(ds - dQ)) <= 1e-11 * np.max(np.abs(dQ))
    # the resting reference state stays at rest
    Qr = np.zeros_like(Q); Qr[..., 0] = cfg["ref_rho"]; Qr[..., 4] = cfg["ref_rhoe"]
    assert np.max(np.abs(o.rhs(Qr)[..., 0:4])) <= 1e-12 * 1.2 * 9.81


# ------------------------------------------------------------------ O13: curl-invariant metric terms
def warped_3d(N=4, ne=(3, 3, 3), amp=0.08, metric_form=1, **kw):
    """Triply periodic box whose nodes are displaced by a smooth periodic field in all three directions."""
    cfg = W.base_params(N=N, ne=ne, hi=(3.0, 3.0, 3.0), bc=(0, 0, 0), geom=0, grav=0.0, **kw)
    X = W.node_coords(cfg)
    k = 2 * np.pi / 3.0
    s = np.sin(k * X[..., 0]) * np.sin(k * X[..., 1]) * np.sin(k * X[..., 2])
    c = np.cos(k * X[..., 0] + 0.3) * np.sin(k * X[..., 1]) * np.cos(k * X[..., 2])
    Y = X.copy()
    Y[..., 0] += amp * s; Y[..., 1] += 0.7 * amp * c; Y[..., 2] += 0.5 * amp * (s - c)
    cfg["geom"] = 2
    cfg["xyz"] = np.ascontiguousarray(np.moveaxis(Y, -1, 0))
    cfg["metric_form"] = metric_form
    return cfg, Y


def _metric_identity(o, om, e):
    D = om.dmat(o.N); Nq = o.Nq
    Ja = o.elem_geometry(e)["Ja"].reshape(Nq, Nq, Nq, 3, 3)          # [k][j][i][d][c]
    r = (np.einsum("im,kjmc->kjic", D, Ja[..., 0, :]) + np.einsum("jm,kmic->kjic", D, Ja[..., 1, :]) +
         np.einsum("km,mjic->kjic", D, Ja[..., 2, :]))
    return np.max(np.abs(r)) / np.max(np.abs(Ja))


def test_curl_invariant_metrics(oracle_mod):
    cfg1, _ = warped_3d(metric_form=1)
    cfg0, _ = warped_3d(metric_form=0)
    o1, o0 = oracle_mod.Oracle(cfg1), oracle_mod.Oracle(cfg0)
    r1 = max(_metric_identity(o1, oracle_mod, e) for e in range(o1.Ne))
    r0 = max(_metric_identity(o0, oracle_mod, e) for e in range(o0.Ne))
    assert r1 <= 1e-13 and r0 >= 1e-6, (r1, r0)                    # the cross-product form fails on a 3-D warp
    # both forms approximate the same analytic metric: they differ by the interpolation error only
    d = max(np.max(np.abs(o1.elem_geometry(e)["Ja"] - o0.elem_geometry(e)["Ja"])) for e in range(o1.Ne))
    assert 1e-12 < d < 5e-3
    # outward sJ n of the two elements at a shared face are equal and opposite (needed for conservation)
    Nq = o1.Nq
    for e in (0, 13):
        g = o1.elem_geometry(e)
        for f in range(6):
            en = o1.neighbour(e, f); gn = o1.elem_geometry(en)
            assert np.max(np.abs(g["sJn"][f] + gn["sJn"][f ^ 1])) <= 1e-13
    # free stream: a uniform moving state has zero tendency on the warped mesh (closure on: zero gradient too)
    cfg1s, Y = warped_3d(metric_form=1, sgs=1)
    os_ = oracle_mod.Oracle(cfg1s)
    one = np.ones(Y.shape[:2])
    Q = W.conserved(cfg1s, 1.1 * one, 12.0 * one, -7.0 * one, 3.0 * one, 288.0 * one, 0 * one, 0 * one)
    dQ = os_.rhs(Q)
    dx = os_.diagnostics(Q)["min_node_dx"]
    Tf = np.array([13.2, 1.1 * 144 + 1e5, 1.1 * 144 + 1e5, 1.1 * 144 + 1e5, 3.6e5 * 12]) / dx
    for v in range(5):
        assert np.max(np.abs(dQ[..., v])) <= 1e-13 * Tf[v], v
    assert np.max(np.abs(oracle_mod.Oracle(dict(cfg1s, metric_form=0)).rhs(Q)[..., 1])) > 1e-8 * Tf[1]


def test_curl_form_on_affine_and_extruded_meshes(oracle_mod):
    """Affine elements (sheared brick): the products X_l dX_m/dxi are polynomials of degree <= N, so the curl form
    reproduces the cross-product form to round-off.  Terrain mesh (y-extruded, degree-N surface): both forms satisfy
    the discrete metric identity; they differ by the aliasing of the degree-(N+1) products only."""
    from test_oracle_wall import sheared_box
    cfg, _ = sheared_box()
    o0 = oracle_mod.Oracle(cfg); o1 = oracle_mod.Oracle(dict(cfg, metric_form=1))
    for e in range(o0.Ne):
        a, b = o0.elem_geometry(e), o1.elem_geometry(e)
        assert np.max(np.abs(a["Ja"] - b["Ja"])) <= 1e-12 * np.max(np.abs(a["Ja"]))
        assert np.array_equal(a["J"], b["J"])
    cfg, _, _ = W.config4(ne=(6, 1, 4), N=4)
    o0 = oracle_mod.Oracle(cfg); o1 = oracle_mod.Oracle(dict(cfg, metric_form=1))
    for e in range(o0.Ne):
        assert _metric_identity(o0, oracle_mod, e) <= 1e-12 and _metric_identity(o1, oracle_mod, e) <= 1e-12
        a, b = o0.elem_geometry(e), o1.elem_geometry(e)
        assert np.max(np.abs(a["Ja"] - b["Ja"])) <= 1e-4 * np.max(np.abs(a["Ja"]))
