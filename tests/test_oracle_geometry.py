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
