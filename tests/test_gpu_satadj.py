"""GPU parity of the saturation-adjusted equation of state (eq. 15; scope row NEXT-4) against the oracle that
tests/test_oracle_satadj.py pins, through the C ABI, element by element.

Tolerance: with condensate p - p_r is a plain difference of two pressures (no R12), each good to a few ulp of p ~ 1e5 Pa.
The two implementations therefore differ by ~ 4 eps p in p', i.e. by 4 eps p / dx_min in the momentum tendencies, whatever
the size of the tendency: the bar is max(1e-11 max|dQ_f|, 8 eps p_max / dx_min) for the momentum fields and 1e-11 elsewhere."""
import numpy as np
import pytest

import workloads as W
from parity_util import RHS_TOL, STEP_TOL, small_config, state_errors

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2110_00853_b200 as pkg
    return pkg


def cloudy(cfg, Q, oracle_mod, factor=1.3):
    """Config-5-shaped state with q_t scaled up so that a layer of the column is supersaturated (cloud)."""
    o = oracle_mod.Oracle(dict(cfg, satadj=0))
    xyz = W.node_coords(cfg)
    rho = Q[..., 0]; u = Q[..., 1:4] / rho[..., None]; q = Q[..., 5] / rho
    cvm = cfg["c_vd"] * (1 - q) + cfg["c_vv"] * q
    T = cfg["T_0"] + (Q[..., 4] / rho - 0.5 * (u ** 2).sum(-1) - cfg["grav"] * xyz[..., 2] - q * cfg["I_v0"]) / cvm
    del o
    return W.conserved(cfg, rho, u[..., 0], u[..., 1], u[..., 2], T, factor * q, xyz[..., 2])


def _errors(dg, do, cfg, pmax, dx):
    errs = []
    for v in range(6):
        tol = RHS_TOL * np.max(np.abs(do[..., v]))
        if v in (1, 2, 3):
            tol = max(tol, 8 * 2.2e-16 * pmax / dx)
        errs.append(np.max(np.abs(dg[..., v] - do[..., v])) / tol)
    return np.array(errs)


@pytest.mark.parametrize("N", [3, 4])
def test_satadj_rhs_parity(P, oracle_mod, N):
    cfg, Q, dt = small_config(5, N=N)
    cfg = dict(cfg, satadj=1)
    Q = cloudy(cfg, Q, oracle_mod)
    o = oracle_mod.Oracle(cfg); g = P.CmDg(cfg)
    Qs = o.lsrk54(Q, dt, 3)
    # the state really has a cloud layer and a clear one
    ql = np.array([o.primitives(Qs[e, 0], z=W.node_coords(cfg)[e, 0, 2], ref=None)["ql"] for e in range(0, o.Ne, 7)])
    assert (ql > 1e-4).any() and (ql == 0).any()
    dg, do = g.to_host(g.rhs(g.to_device(Qs))), o.rhs(Qs)
    dx = o.diagnostics(Qs)["min_node_dx"]
    err = _errors(dg, do, cfg, 1.02e5, dx)
    assert np.all(err <= 1.0), err
    # the condensate matters: the same state under the non-condensing EOS has a visibly different tendency
    d0 = oracle_mod.Oracle(dict(cfg, satadj=0)).rhs(Qs)
    assert np.max(np.abs(d0[..., 3] - do[..., 3])) > 1e-3 * np.max(np.abs(do[..., 3]))
    g.close()


def test_satadj_steps_diagnostics_and_profiles(P, oracle_mod):
    cfg, Q, dt = small_config(5)
    cfg = dict(cfg, satadj=1, richardson=1)
    Q = cloudy(cfg, Q, oracle_mod)
    o = oracle_mod.Oracle(cfg); g = P.CmDg(cfg)
    Qd = g.to_device(Q); g.lsrk_step(Qd, dt, 20)
    Qo = o.lsrk54(Q, dt, 20)
    assert np.all(state_errors(g.to_host(Qd), Qo) <= STEP_TOL)
    dg, do = g.diagnostics(g.to_device(Qo)), o.diagnostics(Qo)
    assert abs(dg["max_wavespeed"] - do["max_wavespeed"]) <= 1e-12 * do["max_wavespeed"]
    Pg, Po = g.profiles(g.to_device(Qo)), o.profiles(Qo)
    assert np.max(np.abs(Pg[:, 5] - Po[:, 5])) <= 1e-12 * np.max(np.abs(Po[:, 5]))     # h_tot uses the adjusted pressure
    assert np.max(np.abs(Pg[:, 7] - Po[:, 7])) <= 1e-12 * np.max(np.abs(Po[:, 7]))     # theta_v
    g.close()


def test_satadj_needs_moisture(P):
    cfg, Q, dt = small_config(3)
    with pytest.raises(P.CmDgError):
        P.CmDg(dict(cfg, satadj=1))


def test_satadj_extreme_states_converge(P, oracle_mod):
    """The kernel's Newton iteration is bracketed (unsaturated T below, all-liquid T above, midpoint when a step leaves the
    bracket) while the oracle runs the paper's plain Newton.  On states far outside the atmospheric range of the other
    tests (215-325 K, 0.25-1.35 kg/m^3, q_t up to 0.08: three quarters of the nodes heavily supersaturated) both must land
    on the same root: no non-finite value, and the pressure-dependent level statistics and the wave speed agree."""
    cfg, Q, dt = small_config(5)
    cfg = dict(cfg, satadj=1)
    xyz = W.node_coords(cfg)
    rng = np.random.default_rng(20211000)
    shp = xyz[..., 2].shape
    T = rng.uniform(215.0, 325.0, shp); rho = rng.uniform(0.25, 1.35, shp); q = rng.uniform(0.0, 0.08, shp)
    u, v, w = (rng.uniform(-5.0, 5.0, shp) for _ in range(3))
    Qx = W.conserved(cfg, rho, u, v, w, T, q, xyz[..., 2])
    o = oracle_mod.Oracle(cfg); g = P.CmDg(cfg)
    ql = np.array([o.primitives(Qx[e, 3], z=xyz[e, 3, 2], ref=None)["ql"] for e in range(o.Ne)])
    assert (ql > 1e-3).mean() > 0.5 and (ql == 0).any()
    Qd = g.to_device(Qx)
    dg, do = g.diagnostics(Qd), o.diagnostics(Qx)
    assert dg["n_nonfinite"] == 0
    assert abs(dg["max_wavespeed"] - do["max_wavespeed"]) <= 1e-12 * do["max_wavespeed"]
    Pg, Po = g.profiles(Qd), o.profiles(Qx)
    for col in (5, 7):                                   # h_tot and theta_v carry the adjusted pressure of every node
        assert np.max(np.abs(Pg[:, col] - Po[:, col])) <= 1e-12 * np.max(np.abs(Po[:, col])), col
    g.close()
