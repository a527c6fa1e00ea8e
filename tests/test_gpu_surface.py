"""GPU parity of the NEXT-4 pieces that the paper defines in closed form -- drag law (eq. A2), prescribed evaporation and
latent heat flux, density-weighted horizontal statistics (eq. B1-B4) -- against the oracle functions that
tests/test_oracle_surface.py pins, through the C ABI, element by element."""
import numpy as np
import pytest

import workloads as W
from parity_util import RHS_TOL, STEP_TOL, rhs_errors, small_config, state_errors
from test_oracle_wall import sheared_box

pytestmark = pytest.mark.gpu

SURF = dict(drag_cd=1.3e-3, lhf_bottom=147.2, evap_bottom=147.2 / 2.5008e6)   # BOMEX sizes; E = LHF / L_v0


@pytest.fixture(scope="module")
def P():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2110_00853_b200 as pkg
    return pkg


def _rhs_check(P, oracle_mod, cfg, Q, dt, steps=3, tuning=None):
    o = oracle_mod.Oracle(cfg); g = P.CmDg(cfg, tuning=tuning)
    Qs = o.lsrk54(Q, dt, steps)
    dg, do = g.to_host(g.rhs(g.to_device(Qs))), o.rhs(Qs)
    err = rhs_errors(dg, do, cfg, Qs, o.diagnostics(Qs)["min_node_dx"])
    g.close()
    return err, dg, do


@pytest.mark.parametrize("k,N,tuning", [(5, 4, None), (5, 3, None), (5, 5, None), (5, 6, None), (5, 4, {"kernel": 7}), (5, 4, {"kernel": 2}),
                                        (3, 4, None), (4, 4, None)])
def test_surface_flux_rhs_parity(P, oracle_mod, k, N, tuning):
    cfg, Q, dt = small_config(k, N=N)
    cfg = dict(cfg, **SURF)
    if k != 5:
        cfg["evap_bottom"] = 0.0 if cfg["nvar"] == 5 else cfg["evap_bottom"]
    if k == 5:
        # a mean wind so that the drag acts on something (config 5 starts from noise around rest; config 4 has its inflow)
        Q = Q.copy(); Q[..., 1] += 6.0 * Q[..., 0]; Q[..., 2] -= 2.5 * Q[..., 0]
        Q[..., 4] += 0.5 * (6.0 ** 2 + 2.5 ** 2) * Q[..., 0]
    err, dg, do = _rhs_check(P, oracle_mod, cfg, Q, dt, tuning=tuning)
    assert np.all(err <= RHS_TOL), err
    # the surface terms are really in the compared tendencies: without them the bottom nodes differ
    o0 = oracle_mod.Oracle(dict(cfg, drag_cd=0.0, lhf_bottom=0.0, evap_bottom=0.0))
    Qs = oracle_mod.Oracle(cfg).lsrk54(Q, dt, 3)
    d0 = o0.rhs(Qs)
    assert np.max(np.abs(d0[..., 4] - do[..., 4])) > 1e-6 * np.max(np.abs(do[..., 4]))
    if k != 3:
        assert np.max(np.abs(d0[..., 1] - do[..., 1])) > 1e-6 * np.max(np.abs(do[..., 1]))


def test_surface_flux_steps(P, oracle_mod):
    cfg, Q, dt = small_config(5)
    cfg = dict(cfg, **SURF)
    Q = Q.copy(); Q[..., 1] += 6.0 * Q[..., 0]; Q[..., 4] += 18.0 * Q[..., 0]
    o = oracle_mod.Oracle(cfg); g = P.CmDg(cfg)
    Qd = g.to_device(Q); g.lsrk_step(Qd, dt, 30)
    Qo = o.lsrk54(Q, dt, 30)
    assert np.all(state_errors(g.to_host(Qd), Qo) <= STEP_TOL)
    # budgets on the GPU result: water and mass grow by E * area * time
    d0, d1 = g.diagnostics(g.to_device(Q)), g.diagnostics(Qd)
    area = (cfg["hi"][0] - cfg["lo"][0]) * (cfg["hi"][1] - cfg["lo"][1])
    assert abs((d1["water"] - d0["water"]) - cfg["evap_bottom"] * area * 30 * dt) < 1e-9 * d0["water"]
    assert abs((d1["mass"] - d0["mass"]) - cfg["evap_bottom"] * area * 30 * dt) < 1e-11 * d0["mass"]


def test_drag_on_an_oblique_wall(P, oracle_mod):
    cfg, xyz = sheared_box(nvar=6)
    cfg = dict(cfg, drag_cd=2.0e-3, evap_bottom=3e-5, lhf_bottom=80.0, shf_bottom=10.0)
    rng = np.random.default_rng(11)
    shape = xyz.shape[:2]
    Q = W.conserved(cfg, 1.1 + 1e-3 * rng.uniform(-1, 1, shape), 5.0 + rng.normal(0, 1, shape), -2.0 + rng.normal(0, 1, shape),
                    rng.normal(0, 1, shape), 295.0 + 0.1 * rng.normal(0, 1, shape), 0.012 + 1e-4 * rng.uniform(-1, 1, shape), xyz[..., 2])
    o = oracle_mod.Oracle(cfg); g = P.CmDg(cfg)
    err = rhs_errors(g.to_host(g.rhs(g.to_device(Q))), o.rhs(Q), cfg, Q, o.diagnostics(Q)["min_node_dx"])
    assert np.all(err <= RHS_TOL), err


def test_setup_rejects_surface_fluxes_without_a_wall(P):
    cfg, Q, dt = small_config(1)
    with pytest.raises(P.CmDgError):
        P.CmDg(dict(cfg, drag_cd=1e-3))
    with pytest.raises(P.CmDgError):
        P.CmDg(dict(small_config(5)[0], drag_cd=-1.0))


@pytest.mark.parametrize("k,N,tuning", [(5, 4, None), (5, 3, None), (3, 4, None), (4, 4, None), (2, 4, None), (5, 4, {"kernel": 2}), (5, 4, {"order_lex": 1})])
def test_profiles_parity(P, oracle_mod, k, N, tuning):
    cfg, Q, dt = small_config(k, N=N)
    o = oracle_mod.Oracle(cfg); g = P.CmDg(cfg, tuning=tuning)
    Qs = o.lsrk54(Q, dt, 5)                                # some flow, so that fluxes and variances are non-trivial
    Pg, Po = g.profiles(g.to_device(Qs)), o.profiles(Qs)
    assert Pg.shape == Po.shape
    assert np.max(np.abs(Pg[:, 0] - Po[:, 0])) <= 1e-12 * cfg["hi"][2]
    assert np.max(np.abs(Pg[:, 1] - Po[:, 1])) <= 1e-13 * np.max(Po[:, 1])
    rho = Qs[..., 0]
    vals = [Qs[..., 1] / rho, Qs[..., 2] / rho, Qs[..., 3] / rho, None, (Qs[..., 5] / rho if cfg["nvar"] == 6 else 0 * rho), None]
    for m in range(6):
        mean_scale = np.max(np.abs(Po[:, 2 + m]))
        # fluctuation scale of phi: means are accurate to eps * max|phi|, second moments to eps * max|phi'|^2-ish sums
        amp = np.max(np.abs(vals[m])) if vals[m] is not None else mean_scale
        assert np.max(np.abs(Pg[:, 2 + m] - Po[:, 2 + m])) <= 1e-12 * max(amp, 1e-300), ("mean", m)
        wamp = np.max(np.abs(vals[2]))
        assert np.max(np.abs(Pg[:, 8 + m] - Po[:, 8 + m])) <= 1e-11 * max(np.max(np.abs(Po[:, 8 + m])), 1e-3 * wamp * amp, 1e-300), ("flux", m)
        assert np.max(np.abs(Pg[:, 14 + m] - Po[:, 14 + m])) <= 1e-11 * max(np.max(np.abs(Po[:, 14 + m])), 1e-300), ("var", m)
    # repeatable bit for bit (fixed summation order)
    assert np.array_equal(Pg, g.profiles(g.to_device(Qs)))
    g.close()


def test_profiles_do_not_disturb_stepping(P, oracle_mod):
    cfg, Q, dt = small_config(5)
    g = P.CmDg(cfg)
    Qa = g.to_device(Q); g.lsrk_step(Qa, dt, 4)
    Qb = g.to_device(Q); g.lsrk_step(Qb, dt, 2); g.profiles(Qb); g.diagnostics(Qb); g.lsrk_step(Qb, dt, 2)
    assert np.array_equal(g.to_host(Qa), g.to_host(Qb))    # the residual buffer used as scratch is dead between steps
    with pytest.raises(P.CmDgError):
        P.cm_dg_profiles(g.ctx, Qb, np.zeros((3, 20)))
