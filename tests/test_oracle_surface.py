"""Pins for the oracle's surface fluxes and horizontal statistics (scope row NEXT-4):

  * aerodynamic drag law on the bottom wall, eq. (A2): n.(rho tau) = -rho C_d |u_p,int| u_p,int with u_p,int the
    wall-parallel velocity at the first layer of interior nodes;
  * prescribed evaporation E = n.(rho d_qv)|sfc and latent heat flux added to SHF in the wall energy flux
    (BOMEX prescribes both);
  * density-weighted horizontal means, vertical eddy fluxes and variances, eq. (B1)-(B4) P:L756-770.

Every expected value is a closed form or an exact budget: a uniform stream over a flat wall has zero tendency except the
lifted wall flux, whose size is (sJ / (w_0 J)) * flux = 2 / (w_0 h_z) * flux on a brick; volume integrals of the tendency
equal flux * wall area exactly; statistics of fields that are polynomials / sinusoids of the horizontal coordinates have
elementary Gauss-Lobatto sums.
"""
import numpy as np

import workloads as W
from test_oracle_wall import ALPHA, sheared_box


def _box(**kw):
    c = W.base_params(N=4, ne=(3, 2, 2), hi=(300.0, 200.0, 100.0), bc=(0, 0, 1), grav=0.0, sgs=0, nvar=6)
    c.update(kw)
    return c


def _uniform(cfg, xyz, u0, rho=1.1, T=295.0, q=0.012):
    one = np.ones(xyz.shape[:2])
    return W.conserved(cfg, rho * one, u0[0] * one, u0[1] * one, u0[2] * one, T * one, q * one, xyz[..., 2])


def test_drag_law_closed_form_on_a_flat_wall(oracle_mod):
    cd = 1.3e-3
    u0 = np.array([6.0, -2.5, 0.0])
    cfg = _box(drag_cd=cd)
    xyz = W.node_coords(cfg)
    Q = _uniform(cfg, xyz, u0)
    ref = oracle_mod.Oracle(_box()).rhs(Q)                      # free slip: a uniform horizontal stream is steady
    T_f = np.max(np.abs(Q[..., 4])) * np.linalg.norm(u0) / W.min_node_spacing(cfg)     # one flux-derivative term (R23)
    assert np.max(np.abs(ref)) < 1e-13 * T_f
    dQ = oracle_mod.Oracle(cfg).rhs(Q) - ref
    N = cfg["N"]; Nq = N + 1; w0 = 2.0 / (N * (N + 1)); hz = 100.0 / cfg["ne"][2]
    lift = 2.0 / (w0 * hz)
    expect = np.zeros_like(dQ)
    Ex, Ey, Ez = cfg["ne"]
    bottom = np.arange(Ex * Ey)                                  # ez = 0 elements, nodes k = 0
    speed = np.linalg.norm(u0)
    for i in range(3):
        expect[bottom, : Nq * Nq, 1 + i] = -lift * 1.1 * cd * speed * u0[i]
    assert np.max(np.abs(dQ - expect)) < 1e-12 * lift * 1.1 * cd * speed ** 2
    # budget: the volume integral of the momentum tendency is -rho C_d |u| u times the wall area
    M = oracle_mod.Oracle(cfg).mass()
    for i in range(2):
        tot = float(np.sum(M * dQ[..., 1 + i]))
        assert abs(tot + 1.1 * cd * speed * u0[i] * 300.0 * 200.0) < 1e-12 * abs(tot)


def test_drag_uses_the_first_interior_layer_and_only_the_wall_parallel_part(oracle_mod):
    cd = 2.0e-3
    cfg = _box(drag_cd=cd)
    xyz = W.node_coords(cfg)
    N = cfg["N"]; Nq = N + 1; NF = Nq * Nq
    Ex, Ey, Ez = cfg["ne"]
    bottom = np.arange(Ex * Ey)
    # velocity differs per nodal layer: (u, v, w) = (2 + k, 1, 0.5 k) in the bottom elements
    rho = 1.2
    Q = _uniform(cfg, xyz, np.array([0.0, 0.0, 0.0]), rho=rho)
    lay = np.repeat(np.arange(Nq), NF).astype(float)             # k of node n
    Y = W.conserved(cfg, rho + 0 * lay, 2.0 + lay, 1.0 + 0 * lay, 0.5 * lay, 295.0 + 0 * lay, 0.012 + 0 * lay, xyz[0, :, 2])
    Q[bottom] = Y[None]
    o_d, o_0 = oracle_mod.Oracle(cfg), oracle_mod.Oracle(_box())
    diff = o_d.rhs(Q) - o_0.rhs(Q)                               # the drag is the only difference
    w0 = 2.0 / (N * (N + 1)); lift = 2.0 / (w0 * (100.0 / Ez))
    up = np.array([3.0, 1.0, 0.0])                               # layer k = 1, the w = 0.5 there is wall-normal: dropped
    for i in range(3):
        got = diff[bottom, :NF, 1 + i]
        assert np.max(np.abs(got + lift * rho * cd * np.linalg.norm(up) * up[i])) < 1e-12 * lift
    assert np.max(np.abs(diff[bottom, NF:, :])) == 0.0          # nothing but the wall nodes
    assert np.max(np.abs(diff[Ex * Ey:])) == 0.0
    assert np.max(np.abs(diff[..., 0])) == 0.0 and np.max(np.abs(diff[..., 4:])) == 0.0


def test_drag_on_an_oblique_wall_is_tangent_to_it(oracle_mod):
    cd = 1.0e-3
    cfg, xyz = sheared_box(nvar=6)
    cfg["sgs"] = 0
    cfg_d = dict(cfg, drag_cd=cd)
    u0 = np.array([7.0, -3.0, 2.0])                              # not tangent to the tilted wall
    Q = _uniform(cfg, xyz, u0)
    diff = oracle_mod.Oracle(cfg_d).rhs(Q) - oracle_mod.Oracle(cfg).rhs(Q)
    o = oracle_mod.Oracle(cfg)
    N = cfg["N"]; Nq = N + 1; w0 = 2.0 / (N * (N + 1))
    nrm = np.array([ALPHA, 0.0, -1.0]) / np.sqrt(1 + ALPHA ** 2)   # outward normal of the bottom wall z = ALPHA x
    up = u0 - (u0 @ nrm) * nrm
    Ex, Ey, Ez = cfg["ne"]
    e = 1 + Ex * 0
    geo = o.elem_geometry(e)
    for n in range(Nq * Nq):
        sJ = np.linalg.norm(geo["Ja"][n][2]); lift = sJ / (w0 * geo["J"][n])
        got = diff[e, n, 1:4]
        # the drag is added to a wall flux of size sJ p ~ 1e8 before the lift: the difference of the two runs carries its ulp
        size = lift * 1.1 * cd * np.linalg.norm(up) ** 2
        assert np.max(np.abs(got + lift * 1.1 * cd * np.linalg.norm(up) * up)) < 1e-9 * size
        assert abs(got @ nrm) < 1e-9 * size                      # no wall-normal force


def test_evaporation_and_latent_heat_budgets(oracle_mod):
    E, lhf, shf = 5.9e-5, 147.2, 9.5                             # BOMEX-like sizes, E = LHF / L_v0
    cfg = _box(evap_bottom=E, lhf_bottom=lhf, shf_bottom=shf, grav=9.81, sgs=1)
    rng = np.random.default_rng(5)
    xyz = W.node_coords(cfg)
    shape = xyz.shape[:2]
    Q = W.conserved(cfg, 1.1 + 1e-3 * rng.uniform(-1, 1, shape), rng.normal(0, 1, shape), rng.normal(0, 1, shape),
                    rng.normal(0, 1, shape), 295.0 + 0.1 * rng.normal(0, 1, shape), 0.012 + 1e-4 * rng.uniform(-1, 1, shape), xyz[..., 2])
    o = oracle_mod.Oracle(cfg)
    dQ = o.rhs(Q); M = o.mass()
    area = 300.0 * 200.0
    for v, flux in ((0, E), (5, E), (4, shf + lhf)):
        tot = float(np.sum(M * dQ[..., v]))
        scale = float(np.sum(M * np.abs(dQ[..., v])))
        assert abs(tot - flux * area) < 1e-12 * scale, (v, tot, flux * area)
    # against the run without surface fluxes only the bottom wall nodes change, by lift * flux
    d = dQ - oracle_mod.Oracle(_box(grav=9.81, sgs=1)).rhs(Q)
    N = cfg["N"]; NF = (N + 1) ** 2; w0 = 2.0 / (N * (N + 1)); lift = 2.0 / (w0 * 50.0)
    Ex, Ey, Ez = cfg["ne"]
    bottom = np.arange(Ex * Ey)
    assert np.max(np.abs(d[bottom, :NF, 0] - lift * E)) < 1e-12 * lift * E + 1e-9 * np.max(np.abs(dQ[..., 0]))
    assert np.max(np.abs(d[bottom, :NF, 5] - lift * E)) < 1e-12 * lift * E + 1e-9 * np.max(np.abs(dQ[..., 5]))
    assert np.max(np.abs(d[bottom, :NF, 4] - lift * (shf + lhf))) < 1e-9 * np.max(np.abs(dQ[..., 4]))
    assert np.max(np.abs(d[bottom, :NF, 1:4])) == 0.0
    assert np.max(np.abs(d[bottom, NF:])) == 0.0 and np.max(np.abs(d[Ex * Ey:])) == 0.0


# ------------------------------------------------------------------ App. B statistics
def test_profiles_of_a_horizontally_uniform_state(oracle_mod):
    cfg = _box(grav=9.81)
    xyz = W.node_coords(cfg)
    z = xyz[..., 2]
    rho = 1.2 - 1e-4 * z; T = 300.0 - 6e-3 * z; q = 0.015 - 1e-5 * z
    Q = W.conserved(cfg, rho, 3.0 + 0.01 * z, -1.0 + 0 * z, 0.2 + 0 * z, T, q, z)
    o = oracle_mod.Oracle(cfg)
    P = o.profiles(Q)
    Nq = cfg["N"] + 1
    assert P.shape == (cfg["ne"][2] * Nq, 20)
    zl = xyz[::cfg["ne"][0] * cfg["ne"][1], ::Nq * Nq, 2].reshape(-1)     # level heights (ez, k)
    assert np.max(np.abs(P[:, 0] - zl)) < 1e-12 * 100.0
    assert np.max(np.abs(P[:, 1] - (1.2 - 1e-4 * zl))) < 1e-14
    assert np.max(np.abs(P[:, 2] - (3.0 + 0.01 * zl))) < 1e-13
    assert np.max(np.abs(P[:, 3] + 1.0)) < 1e-14 and np.max(np.abs(P[:, 4] - 0.2)) < 1e-14
    assert np.max(np.abs(P[:, 6] - (0.015 - 1e-5 * zl))) < 1e-15
    prim = [o.primitives(Q[0, k * Nq * Nq], z=z[0, k * Nq * Nq]) for k in range(Nq)]
    assert np.max(np.abs(P[:Nq, 5] - [p["htot"] for p in prim])) < 1e-15 * 4e5
    assert np.max(np.abs(P[:Nq, 7] - [p["theta_v"] for p in prim])) < 1e-13 * 300.0
    assert np.max(np.abs(P[:, 8:14])) < 1e-12 and np.max(np.abs(P[:, 14:20] / np.maximum(P[:, 2:8] ** 2, 1.0))) < 1e-24


def test_profiles_favre_mean_flux_and_variance_closed_forms(oracle_mod):
    # periodic box, fields that the (N+1)-point Gauss-Lobatto rule integrates exactly (degree <= 2N - 1 = 7 per element):
    # with s = x / Lx in an element-wise polynomial form.  rho = r0 (1 + a X), w = w0 + b X, q = q0 + c X with X a
    # piecewise-linear zero-mean "sawtooth" per element: X = xi (the element's reference coordinate).
    cfg = _box()
    xyz = W.node_coords(cfg)
    Ex = cfg["ne"][0]; hx = 300.0 / Ex
    xi = 2.0 * ((xyz[..., 0] % hx) / hx) - 1.0                  # reference coordinate in x, same in every element
    xi[np.isclose(xi, -1.0) & (np.arange(xi.shape[1]) % 5 == 4)[None, :]] = 1.0   # right end nodes (x % hx wraps to 0)
    r0, a, w0_, b, q0, c = 1.1, 0.2, 0.5, 2.0, 0.012, 0.004
    rho = r0 * (1.0 + a * xi); w = w0_ + b * xi; q = q0 + c * xi
    # moments of xi under the normalised quadrature: <xi> = 0, <xi^2> = 1/3, <xi^3> = 0, <xi^4> = 1/5 (exact for N = 4)
    Q = W.conserved(cfg, rho, 0 * xi, 0 * xi, w, 290.0 + 0 * xi, q, xyz[..., 2])
    P = oracle_mod.Oracle(cfg).profiles(Q)
    m2, m4 = 1.0 / 3.0, 1.0 / 5.0
    mean_rho = r0
    wbar = (w0_ + a * b * m2)                                   # <rho w> / <rho>
    qbar = (q0 + a * c * m2)
    assert np.max(np.abs(P[:, 1] - mean_rho)) < 1e-14
    assert np.max(np.abs(P[:, 4] - wbar)) < 1e-14 and np.max(np.abs(P[:, 6] - qbar)) < 1e-15
    # w' = b (xi - a m2), q' = c (xi - a m2): <rho w' q'> / <rho> = b c <(1 + a xi)(xi - a m2)^2> = b c (m2 - a^2 m2^2)
    k2 = m2 - a * a * m2 * m2
    assert np.max(np.abs(P[:, 8 + 4] - b * c * k2)) < 1e-14 * b * c          # (w'q')bar
    assert np.max(np.abs(P[:, 8 + 2] - b * b * k2)) < 1e-13                 # (w'w')bar as a flux
    assert np.max(np.abs(P[:, 14 + 2] - b * b * k2)) < 1e-13                # (w'^2)bar as a variance: the same number
    assert np.max(np.abs(P[:, 14 + 4] - c * c * k2)) < 1e-14 * c * c
    assert np.max(np.abs(P[:, 2])) == 0.0 and np.max(np.abs(P[:, 14])) == 0.0
    del m4


def test_profiles_weight_by_the_surface_area_element_on_a_warped_mesh(oracle_mod):
    # geom = 1 (terrain-following levels): W = w_i w_j |Ja^3| -- on the sheared brick |Ja^3| is uniform, so use the
    # terrain warp with a surface that is linear in x per element: the levels are tilted planes of known area ratio.
    cfg = W.base_params(N=3, ne=(2, 1, 2), hi=(200.0, 100.0, 100.0), bc=(0, 0, 1), grav=0.0, nvar=5, geom=1)
    Nq = 4
    xs = W.node_coords(dict(cfg, geom=0))[..., 0]
    x_nodes = np.sort(np.unique(np.round(xs, 9)))
    # surface: tent, slope +s on element 0, -s on element 1  -> z_sfc(x) = s * min(x, 200 - x)
    s = 0.4
    line = np.zeros(2 * Nq)
    ex_x = W.node_coords(dict(cfg, geom=0))[:2, :Nq, 0]                # [ex, i]
    zs = s * np.minimum(ex_x, 200.0 - ex_x)                         # [ex, i]
    cfg["zsfc_nodes"] = np.broadcast_to(zs.reshape(1, 1, 2, Nq), (1, Nq, 2, Nq)).copy()
    xyz = W.node_coords(cfg)
    one = np.ones(xyz.shape[:2])
    # rho = 1 on element column 0, 3 on column 1; phi = u = 1 on column 0, 2 on column 1
    col = (np.arange(xyz.shape[0]) % 2)[:, None] * one
    rho = 1.0 + 2.0 * col; u = 1.0 + col
    Q = W.conserved(cfg, rho, u, 0 * one, 0 * one, 300.0 * one, 0 * one, xyz[..., 2])
    P = oracle_mod.Oracle(cfg).profiles(Q)
    # both columns have the same |slope| at every level, hence equal area weights: <rho> = 2, ubar = (1 + 6) / 4
    assert np.max(np.abs(P[:, 1] - 2.0)) < 1e-13 and np.max(np.abs(P[:, 2] - 1.75)) < 1e-13
    # the level's mean height: z = zt + z_sfc (H - zt) / H with <z_sfc> = s * 50
    o = oracle_mod.Oracle(dict(cfg, geom=0))
    zt = o.profiles(Q)[:, 0]
    assert np.max(np.abs(P[:, 0] - (zt + s * 50.0 * (100.0 - zt) / 100.0))) < 1e-11
    # (u'^2)bar: u' = 1 - 1.75 (weight rho = 1) and 2 - 1.75 (weight 3): (0.5625 + 3 * 0.0625) / 4
    assert np.max(np.abs(P[:, 14] - (0.5625 + 0.1875) / 4.0)) < 1e-13
    del x_nodes, line
