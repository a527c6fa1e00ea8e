"""Pins for the oracle's Roe flux (named at P:L256; scope row NEXT-3).  Every expected value follows from the defining
property of Roe's linearisation -- A~ (U+ - U-) = F(U+) - F(U-) exactly for a calorically perfect gas -- and from exact
solutions of the Riemann problem: supersonic states give the pure upwind flux on either side, an isolated contact moving
with the flow is transported by pure upwinding, and a stationary shock that satisfies the Rankine-Hugoniot relations is
kept (F* = F- = F+).  A wrong eigenvector component, wave strength, average or sign breaks at least one of them."""
import numpy as np

import workloads as W
from test_oracle_next import _cfg, _state


def _roe(oracle_mod, **kw):
    cfg = _cfg(sgs=0, riemann=2, nvar=5, grav=0.0)
    cfg.update(kw)
    return cfg, oracle_mod.Oracle(cfg)


def test_roe_consistency_and_conservation(oracle_mod):
    for nvar in (5, 6):
        cfg, o = _roe(oracle_mod, nvar=nvar)
        rng = np.random.default_rng(3)
        for _ in range(10):
            n = rng.normal(0, 1, 3); n /= np.linalg.norm(n)
            Ym = _state(cfg, 1.1 + 0.1 * rng.uniform(), rng.normal(0, 30, 3), 290 + 10 * rng.uniform(), 0.01)
            Yp = _state(cfg, 1.0 + 0.1 * rng.uniform(), rng.normal(0, 30, 3), 285 + 10 * rng.uniform(), 0.012)
            nF = o.flux1(Ym) @ n
            assert np.max(np.abs(o.rusanov(Ym, Ym, n) - nF)) <= 1e-12 * np.max(np.abs(nF))      # F*(Y, Y) = n.F(Y)
            a, b = o.rusanov(Ym, Yp, n), o.rusanov(Yp, Ym, -n)
            assert np.max(np.abs(a + b) / np.maximum(np.abs(a), 1e-3 * np.max(np.abs(a)))) <= 1e-11   # equal and opposite


def test_roe_property_gives_pure_upwinding_for_supersonic_states(oracle_mod):
    # all three wave speeds of one sign: sum_k |lambda_k| alpha_k r_k = +-(F+ - F-) by Roe's property, so F* is the flux of
    # the upwind state -- for ANY pair of states and an oblique normal, with gravity potential and the T_0 energy offset
    cfg, o = _roe(oracle_mod, grav=9.81)
    rng = np.random.default_rng(8)
    for _ in range(10):
        n = rng.normal(0, 1, 3); n /= np.linalg.norm(n)
        t = np.cross(n, [0.3, -0.5, 0.8]); t /= np.linalg.norm(t)
        z = 500.0 * rng.uniform()
        uL = 900.0 * n + 40.0 * rng.normal() * t; uR = 820.0 * n + 40.0 * rng.normal() * t
        YL = _state(cfg, 1.2, uL, 280.0, 0.0, z); YR = _state(cfg, 0.8 + 0.3 * rng.uniform(), uR, 310.0, 0.0, z)
        FL, FR = o.flux1(YL, z) @ n, o.flux1(YR, z) @ n
        assert np.max(np.abs(o.rusanov(YL, YR, n, z) - FL) / np.abs(FL)) <= 2e-12              # everything leaves to the right
        assert np.max(np.abs(o.rusanov(YL, YR, -n, z) + FR) / np.abs(FR)) <= 2e-12             # seen from the other side


def test_roe_moving_contact_and_shear_are_upwinded(oracle_mod):
    cfg, o = _roe(oracle_mod)
    n = np.array([0.0, 0.0, 1.0])
    p = 9.0e4; R = cfg["R_d"]
    # density and tangential-velocity jump, common normal velocity w = 12 m/s and pressure: only the |u_n| waves are
    # excited, F* - F(upwind) = 0 (subsonic!); Rusanov would add (c/2) times the jump
    YL = _state(cfg, 1.2, (3.0, -4.0, 12.0), p / (1.2 * R)); YR = _state(cfg, 0.9, (-7.0, 2.0, 12.0), p / (0.9 * R))
    F, FL = o.rusanov(YL, YR, n), o.flux1(YL) @ n
    assert np.max(np.abs(F - FL) / np.maximum(np.abs(FL), 1.0)) <= 1e-11
    F2, FR = o.rusanov(YL, YR, -n), o.flux1(YR) @ (-n)       # normal reversed: u.n < 0, the upwind state is the "+" one
    assert np.max(np.abs(F2 - FR) / np.maximum(np.abs(FR), 1.0)) <= 1e-11
    orus = oracle_mod.Oracle(dict(cfg, riemann=0))
    assert abs(orus.rusanov(YL, YR, n)[0] - FL[0]) > 10.0


def test_roe_keeps_a_stationary_shock(oracle_mod):
    cfg, o = _roe(oracle_mod)
    g = (cfg["c_vd"] + cfg["R_d"]) / cfg["c_vd"]; R = cfg["R_d"]
    # Rankine-Hugoniot for a normal shock at rest, upstream Mach number M1 (energy measured from T_0: the offset cancels in
    # the jump conditions because the mass flux is continuous)
    M1, rho1, T1 = 2.0, 1.0, 250.0
    c1 = np.sqrt(g * R * T1); u1 = M1 * c1; p1 = rho1 * R * T1
    rho2 = rho1 * (g + 1) * M1 ** 2 / ((g - 1) * M1 ** 2 + 2); u2 = rho1 * u1 / rho2
    p2 = p1 * (1 + 2 * g / (g + 1) * (M1 ** 2 - 1)); T2 = p2 / (rho2 * R)
    n = np.array([1.0, 0.0, 0.0])
    YL = _state(cfg, rho1, (u1, 0, 0), T1); YR = _state(cfg, rho2, (u2, 0, 0), T2)
    FL, FR = o.flux1(YL) @ n, o.flux1(YR) @ n
    scale = np.maximum(np.abs(FL), 1.0)
    assert np.max(np.abs(FL - FR) / scale) <= 1e-13           # the two states do satisfy the jump conditions
    assert abs(YL[0] - YR[0]) > 1.0 and abs(u1 - u2) > 300.0  # and it is a strong shock
    F = o.rusanov(YL, YR, n)
    assert np.max(np.abs(F - FL) / scale) <= 1e-12


def test_roe_on_the_mesh_conserves_and_keeps_walls_closed(oracle_mod):
    cfg, Q, dt = W.config3(ne=(3, 2, 3), N=3, hi=(600.0, 400.0, 562.5))
    cfg = dict(cfg, riemann=2, shf_bottom=0.0)
    o = oracle_mod.Oracle(cfg)
    rng = np.random.default_rng(9)
    Q = Q.copy(); Q[..., 1:4] += rng.normal(0, 0.5, Q[..., 1:4].shape)
    dQ = o.rhs(Q); M = o.mass()
    for v in (0, 4):
        assert abs(np.sum(M * dQ[..., v])) <= 1e-12 * np.sum(M * np.abs(dQ[..., v])), v
    assert np.max(np.abs(o.rhs(Q, form="strong") - dQ)) <= 1e-11 * np.max(np.abs(dQ))
    Qr = np.zeros_like(Q); Qr[..., 0] = cfg["ref_rho"]; Qr[..., 4] = cfg["ref_rhoe"]
    assert np.max(np.abs(o.rhs(Qr)[..., 0:4])) <= 1e-12 * 1.2 * 9.81       # the resting reference state stays at rest
