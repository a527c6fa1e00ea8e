"""Pins for O2 (mesh, terrain warp, metric terms, face normals, mass) of the oracle.

Fixed by geometry itself: volumes and areas of the mesh, closedness of each element's surface, equal and
opposite face vectors on shared faces, the discrete metric identity, and J^-1 being the inverse of the
numerically differentiated mapping (eq. 24).
"""
import numpy as np
import pytest

import workloads as W


def _warped_cfg(N=4, ne=(6, 1, 4)):
    cfg, Q, dt = W.config4(ne=ne, N=N)
    return cfg


def _general_cfg(N=3, ne=(3, 3, 2)):
    """geom=2: a y-extruded warp given through explicit coordinates (exercises the xyz input path)."""
    cfg = W.base_params(N=N, ne=ne, hi=(3.0, 2.0, 1.5), bc=(0, 0, 1), geom=0)
    xyz = W.node_coords(cfg)
    x, z = xyz[..., 0].copy(), xyz[..., 2].copy()
    xyz[..., 2] = z + 0.15 * np.sin(2 * np.pi * x / 3.0) * (1.5 - z) / 1.5
    cfg["geom"] = 2
    cfg["xyz"] = np.ascontiguousarray(np.moveaxis(xyz, -1, 0))   # [3][Ne][Np]
    return cfg


def test_coords_match_generator(oracle_mod):
    for cfg in (W.config1()[0], _warped_cfg(), _general_cfg()):
        o = oracle_mod.Oracle(cfg)
        x = o.coords()
        ref = W.node_coords(cfg) if cfg["geom"] != 2 else np.moveaxis(cfg["xyz"], 0, -1)
        scale = np.max(np.abs(ref))
        assert np.max(np.abs(x - ref)) < 1e-13 * scale


def test_flat_metrics(oracle_mod):
    cfg = W.base_params(N=4, ne=(3, 2, 4), lo=(-1.0, 0.5, 0.0), hi=(2.0, 2.5, 6.0))
    o = oracle_mod.Oracle(cfg)
    hx, hy, hz = 1.0, 1.0, 1.5
    xi, w = oracle_mod.lgl(4)
    for e in (0, 5, o.Ne - 1):
        g = o.elem_geometry(e)
        assert np.max(np.abs(g["J"] - hx * hy * hz / 8)) < 1e-14
        Ja = g["Ja"]
        want = np.diag([hy * hz / 4, hx * hz / 4, hx * hy / 4])
        assert np.max(np.abs(Ja - want[None])) < 1e-14
        assert np.max(np.abs(g["lift"][0] - (2 / hx) / w[0])) < 1e-12
        assert np.max(np.abs(g["lift"][5] - (2 / hz) / w[0])) < 1e-12
        assert np.allclose(g["sJn"][0][..., 0], -hy * hz / 4) and np.allclose(g["sJn"][3][..., 1], hx * hz / 4)
    assert abs(o.mass().sum() - 3.0 * 2.0 * 6.0) < 1e-12


def test_flat_metrics_far_from_the_origin(oracle_mod):
    """Eq. (24), on a flat brick that sits where config 4's last elements sit: 2.9e5 m from the origin in x
    (and 1.2e5 m in y), 2500 m x 700 m elements, N = 4.  D annihilates constants, so differentiating the coordinates
    relative to the element's first node is eq. (24) unchanged; in floating point it is not: products D_im x_m that carry
    the offset leave sum_m D_im x_m = x * (rounding of the row sum of D) ~ 3e5 * 1e-16 where the exact derivative is 0, i.e.
    spurious off-diagonal metric terms of relative size ~ eps |x| / h and a free-stream residual of the same size.
    Pinned here (measured with the element-relative form / with absolute coordinates, i.e. with the `- x[d]` terms of
    elem_geo_compute removed; the second column fails):
      off-diagonal Ja entries  <= 32 eps max|Ja_dd|        6.6 eps  / 1270 eps
      uniform-flow tendency    <  1e-13 T_f per field      4.8e-15  / 8.4e-13
    The diagonal entries and J meet their closed forms to 16 eps |x| / h (the nodal coordinates themselves are rounded at
    ulp(3e5) = 6e-11 on a 700 m element, which no differentiation can undo)."""
    hx, hy, hz = 2500.0, 2500.0, 700.0
    lo = (2.9e5, 1.2e5, 0.0)
    cfg = W.base_params(N=4, ne=(4, 2, 3), lo=lo, hi=(lo[0] + 4 * hx, lo[1] + 2 * hy, 3 * hz), bc=(0, 0, 0), grav=0.0)
    o = oracle_mod.Oracle(cfg)
    eps = np.finfo(float).eps
    want = np.array([hy * hz / 4, hx * hz / 4, hx * hy / 4])
    off = ~np.eye(3, dtype=bool)
    rel = 16 * eps * (lo[0] + 4 * hx) / hz
    for e in range(o.Ne):
        g = o.elem_geometry(e)
        assert np.max(np.abs(g["Ja"][:, off])) <= 32 * eps * want.max(), e
        for d in range(3):
            assert np.max(np.abs(g["Ja"][:, d, d] - want[d])) <= rel * want[d], (e, d)
        assert np.max(np.abs(g["J"] - hx * hy * hz / 8)) <= rel * hx * hy * hz / 8, e
    z = o.coords()[..., 2]
    one = np.ones_like(z)
    Q = W.conserved(cfg, 1.1 * one, 12.0 * one, -7.0 * one, 3.0 * one, 288.0 * one, 0.0 * one, z)
    dx = o.diagnostics(Q)["min_node_dx"]
    for form in ("weak", "strong"):
        dQ = o.rhs(Q, form)
        for v in range(cfg["nvar"]):
            Tf = max(abs(np.array(o.flux1(Q[0, 0])[v]).max()), 1e-300) / dx
            assert np.max(np.abs(dQ[..., v])) < 1e-13 * Tf, (form, v)


@pytest.mark.parametrize("maker", [_warped_cfg, _general_cfg])
def test_warped_metrics(oracle_mod, maker):
    cfg = maker()
    o = oracle_mod.Oracle(cfg)
    N = cfg["N"]; Nq = N + 1
    xi, w = oracle_mod.lgl(N)
    D = oracle_mod.dmat(N)
    x = o.coords()
    I = np.eye(Nq)
    Dr = np.kron(I, np.kron(I, D)); Ds = np.kron(I, np.kron(D, I)); Dt = np.kron(D, np.kron(I, I))
    total_mass = 0.0
    for e in range(o.Ne):
        g = o.elem_geometry(e)
        # (i) Ja / J is the inverse of the differentiated mapping dx/dxi
        dxdxi = np.stack([Dr @ x[e], Ds @ x[e], Dt @ x[e]], axis=1)        # [n, d, c] = d x_c / d xi_d
        for n in range(o.Np):
            a = g["Ja"][n] / g["J"][n]                                      # a[d, c] = d xi_d / d x_c
            assert np.max(np.abs(dxdxi[n].T @ a - np.eye(3))) < 1e-12      # sum_d (dx_c'/dxi_d)(dxi_d/dx_c)
            assert abs(np.linalg.det(dxdxi[n]) - g["J"][n]) < 1e-12 * abs(g["J"][n])
        assert np.all(g["J"] > 0)
        # (ii) discrete metric identity: sum_d D_d (Ja^d_c) = 0 (free-stream preservation, R4)
        scale = np.max(np.abs(g["Ja"]))
        for c in range(3):
            r = Dr @ g["Ja"][:, 0, c] + Ds @ g["Ja"][:, 1, c] + Dt @ g["Ja"][:, 2, c]
            assert np.max(np.abs(r)) < 1e-12 * scale * Nq * Nq
        # (iii) closed surface: sum over faces of w_a w_b sJ n = 0
        wf = np.outer(w, w)   # [b, a]
        tot = sum((g["sJn"][f] * wf[..., None]).sum(axis=(0, 1)) for f in range(6))
        assert np.max(np.abs(tot)) < 1e-12 * scale
        total_mass += g["M"].sum()
        # (iv) the face vector seen from the neighbour is equal and opposite
        for f in range(6):
            en = o.neighbour(e, f)
            if en < 0:
                continue
            gn = o.elem_geometry(en)
            assert np.max(np.abs(g["sJn"][f] + gn["sJn"][f ^ 1])) < 1e-12 * scale
            assert np.max(np.abs(g["lift"][f] * g["J"].reshape(Nq, Nq, Nq)[_face(f, Nq)] -
                                 gn["lift"][f ^ 1] * gn["J"].reshape(Nq, Nq, Nq)[_face(f ^ 1, Nq)])) < 1e-10 * scale
    # (v) total volume: exact for the degree-N interpolated surface
    if cfg["geom"] == 1:
        Ex, Ey, Ez = cfg["ne"]
        hx = cfg["hi"][0] / Ex; Ly = cfg["hi"][1]; H = cfg["hi"][2]
        zs = np.asarray(cfg["zsfc_nodes"])[0].reshape(Ex, Nq)
        vol = Ly * np.sum(w[None, :] * (hx / 2) * (H - zs))
        assert abs(total_mass - vol) < 1e-12 * vol
    else:
        assert abs(total_mass - 3.0 * 2.0 * 1.5) < 0.2   # sine warp: not exact, only a sanity bound


def _face(f, Nq):
    d = f // 2; at = (Nq - 1) if f % 2 else 0
    idx = [slice(None)] * 3          # array is [k, j, i]
    idx[2 - d] = at
    return tuple(idx)


def test_neighbours_periodic_and_wall(oracle_mod):
    cfg = W.base_params(N=2, ne=(3, 2, 2), bc=(0, 0, 1))
    o = oracle_mod.Oracle(cfg)
    # element (0,0,0)
    assert o.neighbour(0, 0) == 2 and o.neighbour(0, 1) == 1          # x periodic
    assert o.neighbour(0, 2) == 3 and o.neighbour(0, 3) == 3          # y periodic, Ey=2
    assert o.neighbour(0, 4) == -1 and o.neighbour(0, 5) == 6         # z wall / interior
    assert o.neighbour(6, 5) == -1
