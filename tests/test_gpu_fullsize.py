"""GPU parity at the sizes BASELINE.json names (rows g1 / g2 of the scope table): configs 2, 3, 4 in full, element by
element; config 5 stepped 100 times on the 12x12x6 cut SURVEY 8(d) names; config 5 at full size (and the N = 3, 5, 6
meshes of the order sweep) on sampled element columns, for one RHS and for one whole fused LSRK54 step (stage kernels
MODE 2 and MODE 1).  Tolerances are BASELINE.json's: 1e-11 per field for one RHS, 1e-9 after 100 steps (reading R19)."""
import numpy as np
import pytest

import workloads as W
from parity_util import RHS_TOL, STEP_TOL, rhs_errors, state_errors

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2110_00853_b200 as pkg
    return pkg


@pytest.mark.parametrize("k", [2, 3, 4])
def test_full_size_rhs_and_100_steps(P, oracle_mod, k):
    """BASELINE configs 2 (40x1x20), 3 (32x32x16), 4 (120x1x30) at their stated sizes: one RHS at t = 0, 100 fused
    LSRK54 steps, and one RHS on the oracle's 100-step state, every element and node compared."""
    cfg, Q, dt = W.CONFIGS[k]()
    o = oracle_mod.Oracle(cfg)
    g = P.CmDg(cfg)
    dx = o.diagnostics(Q)["min_node_dx"]
    err = rhs_errors(g.to_host(g.rhs(g.to_device(Q))), o.rhs(Q), cfg, Q, dx)
    assert np.all(err <= RHS_TOL), ("t0", err)
    Qd = g.to_device(Q)
    g.lsrk_step(Qd, dt, 100)
    Qo = o.lsrk54(Q, dt, 100)
    err = state_errors(g.to_host(Qd), Qo)
    assert np.all(err <= STEP_TOL), ("100 steps", err)
    err = rhs_errors(g.to_host(g.rhs(g.to_device(Qo))), o.rhs(Qo), cfg, Qo, dx)
    assert np.all(err <= RHS_TOL), ("stepped", err)
    g.close()


def test_config2_1000_steps(P, oracle_mod):
    """Config 2 as BASELINE states it: 1000 LSRK54 steps.  The parity bar is defined at step 100 (previous test); here the
    same comparison is continued to step 1000 with the tolerance scaled by the step count, and mass / energy must stay
    conserved to round-off on the CUDA path (free-slip walls, periodic sides)."""
    cfg, Q, dt = W.config2()
    o = oracle_mod.Oracle(cfg)
    g = P.CmDg(cfg)
    Qd = g.to_device(Q)
    d0 = g.diagnostics(Qd)
    g.lsrk_step(Qd, dt, 1000)
    d1 = g.diagnostics(Qd)
    Qo = o.lsrk54(Q, dt, 1000)
    err = state_errors(g.to_host(Qd), Qo)
    assert np.all(err <= 10 * STEP_TOL), err
    assert d1["n_nonfinite"] == 0
    for key in ("mass", "energy"):
        assert abs(d1[key] - d0[key]) <= 1e-12 * abs(d0[key]), (key, d0[key], d1[key])
    g.close()


def test_config5_cut_100_steps(P, oracle_mod):
    """Config 5 on the 12x12x6-element cut of the same profiles: 100 fused steps and the RHS after them."""
    cfg, Q, dt = W.config5(ne=(12, 12, 6), N=4, hi=(750.0, 750.0, 3000.0))
    o = oracle_mod.Oracle(cfg)
    g = P.CmDg(cfg)
    Qd = g.to_device(Q)
    g.lsrk_step(Qd, dt, 100)
    Qo = o.lsrk54(Q, dt, 100)
    err = state_errors(g.to_host(Qd), Qo)
    assert np.all(err <= STEP_TOL), err
    err = rhs_errors(g.to_host(g.rhs(g.to_device(Qo))), o.rhs(Qo), cfg, Qo, o.diagnostics(Qo)["min_node_dx"])
    assert np.all(err <= RHS_TOL), err
    g.close()


def _columns(g, T, cols, Ex, Ey, Ez):
    """Rows of the device array T[nv, stride] for the element columns (cx, cy) -> list of [Ez, Np, nv] host arrays."""
    import torch
    pos_of_lex = np.empty(g.n_elem, dtype=np.int64)
    pos_of_lex[g.lex_of_elem] = np.arange(g.n_elem)
    out = []
    for cx, cy in cols:
        full = cx + Ex * (cy + Ey * np.arange(Ez))
        idx = (pos_of_lex[full][:, None] * g.np + np.arange(g.np)[None, :]).reshape(-1)
        out.append(T[:, torch.from_numpy(idx).to(T.device)].cpu().numpy().T.reshape(Ez, g.np, T.shape[0]))
    return out


def _sub_brick(Q, cx, cy, R, Ex, Ey, Ez):
    sx = (cx + np.arange(-R, R + 1)) % Ex
    sy = (cy + np.arange(-R, R + 1)) % Ey
    lex = (sx[None, None, :] + Ex * (sy[None, :, None] + Ey * np.arange(Ez)[:, None, None])).reshape(-1)
    W_ = 2 * R + 1
    centre = R + W_ * (R + W_ * np.arange(Ez))
    return np.ascontiguousarray(Q[lex]), centre


@pytest.mark.parametrize("N", [3, 5, 6])
def test_order_sweep_full_size_sampled_rhs(P, oracle_mod, N):
    """The N = 3, 5, 6 meshes of the fixed-DOF sweep (~55 M nodes each) in the launch configuration bench.py times:
    cm_dg_rhs on the whole mesh against the oracle on the 5x5xEz sub-brick around sampled columns (the RHS of an
    element depends on its 2-ring; the lateral closure of the sub-brick is not seen by the centre column)."""
    Ex, Ey, Ez = W.SWEEP5[N]
    cfg, Q, dt = W.config5(ne=(Ex, Ey, Ez), N=N, hi=(6000.0, 6000.0, 3000.0))     # the same 6 km x 6 km x 3 km box at every order
    g = P.CmDg(cfg)
    dQd = g.rhs(g.to_device(Q))
    sub_cfg, _, _ = W.config5(ne=(5, 5, Ez), N=N, hi=(5 * 6000.0 / Ex, 5 * 6000.0 / Ey, 3000.0))
    o = oracle_mod.Oracle(sub_cfg)
    cols = ((0, 0), (Ex // 2 - 1, Ey // 2 + 2), (Ex - 1, Ey - 1))
    for (cx, cy), got in zip(cols, _columns(g, dQd, cols, Ex, Ey, Ez)):
        Qs, centre = _sub_brick(Q, cx, cy, 2, Ex, Ey, Ez)
        dQo = o.rhs(Qs)
        for v in range(g.nvar):
            err = np.max(np.abs(got[..., v] - dQo[centre][..., v])) / np.max(np.abs(dQo[..., v]))
            assert err <= RHS_TOL, (N, cx, cy, v, err)
    g.close()


def test_full_size_sampled_fused_step(P, oracle_mod):
    """One whole fused LSRK54 step (stage kernels MODE 2 then MODE 1, three-buffer ring) on the full config-5 mesh,
    element by element on sampled columns.  Five stages widen the domain of dependence to the 10-ring, so the oracle
    steps the 21x21x48 sub-brick around the column; the increment Q(dt) - Q(0) of the centre column is compared."""
    cfg, Q, dt = W.config5()
    Ex, Ey, Ez = cfg["ne"]
    g = P.CmDg(cfg)
    Qd = g.to_device(Q)
    g.lsrk_step(Qd, dt, 1)
    R = 10
    sub_cfg, _, _ = W.config5(ne=(2 * R + 1, 2 * R + 1, Ez), N=cfg["N"], hi=((2 * R + 1) * 6000.0 / Ex, (2 * R + 1) * 6000.0 / Ey, 3000.0))
    o = oracle_mod.Oracle(sub_cfg)
    # one column from every class of position inside the library's element tiles (x-chunks of 32 = one row sweep, y-patches
    # of 16): row start / middle / end x patch bottom / top, spread over different tiles and the periodic wrap
    cols = ((0, 0), (32, 15), (15, 16), (47, 31), (31, 32), (95, 95))
    assert {(cx % 32, cy % 16) for cx, cy in cols} == {(a, b) for a in (0, 15, 31) for b in (0, 15)}
    for (cx, cy), got in zip(cols, _columns(g, Qd, cols, Ex, Ey, Ez)):
        Qs, centre = _sub_brick(Q, cx, cy, R, Ex, Ey, Ez)
        Qo = o.lsrk54(Qs, dt, 1)
        for v in range(g.nvar):
            inc_o = Qo[centre][..., v] - Qs[centre][..., v]
            inc_g = got[..., v] - Qs[centre][..., v]
            err = np.max(np.abs(inc_g - inc_o)) / np.max(np.abs(Qo[..., v] - Qs[..., v]))
            assert err <= STEP_TOL, (cx, cy, v, err)
    g.close()


def test_config5_full_mesh_every_element(P, oracle_mod):
    """BASELINE config 5 at its full size, every one of the 442 368 elements: cm_dg_rhs on the whole mesh against the oracle
    on the whole mesh (about 10 s on 16 host cores), 1e-11 per field.  Needs roughly 25 GB of host memory for the oracle's
    geometry and gradient arrays beside the state copies; on a box with less, the sampled comparison
    (test_gpu_parity.py::test_full_size_sampled_parity) is the one that ran, and this test says so and skips."""
    import psutil
    avail = psutil.virtual_memory().available
    if avail < 48e9:
        print("config 5 full mesh: SAMPLED branch only (%.0f GB of host memory available, 48 GB wanted)" % (avail / 1e9))
        pytest.skip("not enough host memory for the whole-mesh oracle run; the sampled test covers config 5")
    cfg, Q, dt = W.config5()
    g = P.CmDg(cfg)
    got = g.to_host(g.rhs(g.to_device(Q)))
    g.close()
    o = oracle_mod.Oracle(cfg)
    dQo = o.rhs(Q)
    assert dQo.shape == got.shape == (96 * 96 * 48, 125, 6)
    errs = []
    for v in range(6):
        errs.append(np.max(np.abs(got[..., v] - dQo[..., v])) / np.max(np.abs(dQo[..., v])))
    print("config 5 full mesh: FULL branch, all %d elements, max rel err per field %r" % (got.shape[0], errs))
    assert max(errs) <= RHS_TOL, errs
