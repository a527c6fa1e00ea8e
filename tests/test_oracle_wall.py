"""Pins for the BR1 boundary value on an OBLIQUE free-slip wall (App. A3, eq. A6-A8): the branch of the
oracle's gradient that config 4's terrain wall exercises with the closure on.  A sheared brick (geom = 2, planar tilted
bottom and lid, affine elements) makes the wall normal non-axis-aligned while the exact answers stay elementary.

  * a linear velocity field TANGENT to the tilted walls has n.u = 0 there, so u* = u^- - (n.u^-) n = u^- and the BR1
    gradient must be the analytic constant gradient in the wall elements too (an axis normal in place of the true one,
    a wrong sign or a missing projection all leave a lifted jump);
  * a uniform velocity that is NOT tangent has zero volume derivative, so at a wall-face node the gradient is exactly the
    lifted jump  (sJ / (w_0 J)) n_c (u* - u^-)_i = -(sJ / (w_0 J)) (n.u) n_i n_c  with n = -+Ja^3 / |Ja^3| built from the
    mesh geometry -- the statement u* = u - (n.u) n itself; scalars (h_tot, q_t) keep s* = s^- (A8): zero gradient.
"""
import numpy as np

import workloads as W

ALPHA = 0.3     # slope dz/dx of the walls


def sheared_box(N=4, ne=(3, 2, 3), nvar=5):
    cfg = W.base_params(N=N, ne=ne, hi=(300.0, 200.0, 150.0), bc=(0, 0, 1), geom=0, grav=0.0, use_ref=0, sgs=1, nvar=nvar)
    xyz = W.node_coords(cfg).copy()
    xyz[..., 2] += ALPHA * xyz[..., 0]
    cfg["geom"] = 2
    cfg["xyz"] = np.ascontiguousarray(np.moveaxis(xyz, -1, 0))
    # the shear makes the x-ends non-matching for a periodic wrap of z(x); walls in x as well keep the test self-contained
    cfg["bc"] = (1, 0, 1)
    return cfg, xyz


def test_tangent_linear_field_has_exact_gradient_in_wall_elements(oracle_mod):
    cfg, xyz = sheared_box()
    o = oracle_mod.Oracle(cfg)
    x, y, z = xyz[..., 0], xyz[..., 1], xyz[..., 2]
    t = np.array([1.0, 0.0, ALPHA]) / np.sqrt(1.0 + ALPHA ** 2)          # tangent to the tilted walls, in the x-z plane
    a, b, c = 4.0, 2e-2, 0.0                                            # no y-dependence: y is periodic
    s = z - ALPHA * x                                                   # constant on each tilted wall
    amp = a + b * s + c * y
    vel = [t[i] * amp for i in range(3)]
    Q = W.conserved(cfg, np.ones_like(x), *vel, 300.0 + 0 * x, 0 * x, z)
    G = o.gradient(Q)
    grad_amp = np.array([-b * ALPHA, c, b])
    Ex, Ey, Ez = cfg["ne"]
    # elements that touch a tilted wall but not an x-wall (the x-walls are not tangent to this field)
    wall_elems = [ex + Ex * (ey + Ey * ez) for ez in (0, Ez - 1) for ey in range(Ey) for ex in range(1, Ex - 1)]
    for i in range(3):
        for cc in range(3):
            assert np.max(np.abs(G[wall_elems, :, i, cc] - t[i] * grad_amp[cc])) < 1e-13, (i, cc)


def test_wall_value_is_the_tangential_projection(oracle_mod):
    cfg, xyz = sheared_box(nvar=6)
    o = oracle_mod.Oracle(cfg)
    x, z = xyz[..., 0], xyz[..., 2]
    u0 = np.array([7.0, -3.0, 2.0])
    one = np.ones_like(x)
    Q = W.conserved(cfg, 1.1 * one, u0[0] * one, u0[1] * one, u0[2] * one, 295.0 * one, 0.01 * one, 0 * z)
    G = o.gradient(Q)
    N = cfg["N"]; Nq = N + 1
    w0 = 2.0 / (N * (N + 1))
    Ex, Ey, Ez = cfg["ne"]
    for ez, k, sgn in ((0, 0, -1.0), (Ez - 1, N, 1.0)):                   # bottom wall (outward -Ja^3), lid (+Ja^3)
        e = 1 + Ex * (0 + Ey * ez)                                      # not on an x-wall
        geo = o.elem_geometry(e)
        for j in range(Nq):
            for i in range(1, N):                                       # nodes of the zeta face that lie on no other wall
                n = i + Nq * (j + Nq * k)
                A = sgn * geo["Ja"][n][2]                               # sJ n
                sJ = np.linalg.norm(A); nrm = A / sJ
                assert abs(abs(nrm[0]) - ALPHA / np.sqrt(1 + ALPHA ** 2)) < 1e-12   # the wall really is oblique
                lift = sJ / (w0 * geo["J"][n])
                un = float(nrm @ u0)
                for a in range(3):
                    for c in range(3):
                        expect = lift * nrm[c] * (-un * nrm[a])
                        assert abs(G[e, n, a, c] - expect) < 1e-12 * lift * np.linalg.norm(u0), (ez, n, a, c)
                assert np.max(np.abs(G[e, n, 3:5, :])) < 1e-9                  # scalars: s* = s^- (h_tot ~ 3e5 J/kg)
    # away from every wall the gradient of a uniform state vanishes
    e = 1 + Ex * (0 + Ey * 1)
    assert np.max(np.abs(G[e, :, 0:3, :])) < 1e-12
