"""Pins for O3 (thermodynamics, R12 pressure perturbation), O5 (Smagorinsky-Lilly), O6 (fluxes) and
O8 (Rusanov flux, wall ghost state) of the oracle, checked pointwise against what the paper's equations
and elementary gas dynamics fix.
"""
from decimal import Decimal, getcontext

import numpy as np
import pytest

import workloads as W


@pytest.fixture(scope="module")
def dry(oracle_mod):
    return oracle_mod.Oracle(W.base_params(N=2, ne=(1, 1, 1), nvar=5))


@pytest.fixture(scope="module")
def moist(oracle_mod):
    return oracle_mod.Oracle(W.base_params(N=2, ne=(1, 1, 1), nvar=6))


def test_textbook_ideal_gas_limit(oracle_mod):
    """T_0 = 0, g = 0, dry: p = (gamma - 1) rho e_int and c = sqrt(gamma p / rho)."""
    cfg = W.base_params(N=2, ne=(1, 1, 1), T_0=0.0, grav=0.0)
    o = oracle_mod.Oracle(cfg)
    rho, u, v, w, T = 1.1, 3.0, -2.0, 0.5, 290.0
    eint = cfg["c_vd"] * T
    Y = np.array([rho, rho * u, rho * v, rho * w, rho * (eint + 0.5 * (u * u + v * v + w * w))])
    P = o.primitives(Y)
    gamma = (cfg["c_vd"] + cfg["R_d"]) / cfg["c_vd"]
    assert abs(P["p"] - (gamma - 1) * rho * eint) < 1e-9
    assert abs(P["T"] - T) < 1e-11
    assert abs(P["c"] - np.sqrt(gamma * P["p"] / rho)) < 1e-11
    assert abs(P["htot"] - (Y[4] + P["p"]) / rho) < 1e-9
    assert P["pp"] == P["p"]


def test_moist_thermodynamics_roundtrip(moist):
    """State built from (rho, u, T, q) by eq. (6)-(10) returns the same T; p = rho R_m T (eq. 13-14)."""
    cfg = moist.cfg
    rho, T, q, z = 1.05, 288.3, 0.014, 750.0
    u = np.array([4.0, -1.0, 0.3])
    Y = W.conserved(cfg, np.float64(rho), *u, np.float64(T), np.float64(q), np.float64(z))
    P = moist.primitives(Y, z=z)
    Rm = cfg["R_d"] * (1 - q) + cfg["R_v"] * q
    cvm = cfg["c_vd"] * (1 - q) + cfg["c_vv"] * q
    assert abs(P["T"] - T) < 1e-10
    assert abs(P["p"] - rho * Rm * T) < 1e-8
    assert abs(P["q"] - q) < 1e-16
    assert abs(P["c"] - np.sqrt((1 + Rm / cvm) * Rm * T)) < 1e-11
    # internal energy of eq. (7)-(8): (1-q) c_vd (T-T0) + q (c_vv (T-T0) + I_v0)
    I = (1 - q) * cfg["c_vd"] * (T - cfg["T_0"]) + q * (cfg["c_vv"] * (T - cfg["T_0"]) + cfg["I_v0"])
    assert abs(Y[4] / rho - (I + 0.5 * u @ u + cfg["grav"] * z)) < 1e-9


def _exact_pressure(cfg, Y, z, nvar):
    """EOS pressure in 50-digit decimal arithmetic straight from eq. (6)-(14)."""
    getcontext().prec = 50
    D = Decimal
    rho, mu, mv, mw, re = (D(float(v)) for v in Y[:5])
    rq = D(float(Y[5])) if nvar == 6 else D(0)
    q = rq / rho
    cvm = D(cfg["c_vd"]) * (1 - q) + D(cfg["c_vv"]) * q
    Rm = D(cfg["R_d"]) * (1 - q) + D(cfg["R_v"]) * q
    eint = re / rho - (mu * mu + mv * mv + mw * mw) / (2 * rho * rho) - D(cfg["grav"]) * D(float(z))
    T = D(cfg["T_0"]) + (eint - q * D(cfg["I_v0"])) / cvm
    return rho * Rm * T


@pytest.mark.parametrize("nvar", [5, 6])
def test_pressure_perturbation_R12(oracle_mod, nvar):
    """p' of reading R12 equals p - p_r evaluated exactly, to ~1e-13 Pa; p' == 0 bitwise at the reference."""
    cfg = W.base_params(N=2, ne=(1, 1, 1), nvar=nvar)
    o = oracle_mod.Oracle(cfg)
    rng = np.random.default_rng(7)
    worst = 0.0
    for _ in range(200):
        z = rng.uniform(0, 3000)
        rho_r = rng.uniform(0.8, 1.2); T_r = rng.uniform(270, 300); q_r = rng.uniform(0.004, 0.017) if nvar == 6 else 0.0
        Yr = W.conserved(cfg, np.float64(rho_r), 0.0, 0.0, 0.0, np.float64(T_r), np.float64(q_r), np.float64(z))
        rho = rho_r * (1 + 1e-4 * rng.normal()); T = T_r + 0.3 * rng.normal()
        q = q_r + 1e-5 * rng.normal() if nvar == 6 else 0.0
        u = rng.normal(0, 2.0, 3)
        Y = W.conserved(cfg, np.float64(rho), *u, np.float64(T), np.float64(q), np.float64(z))
        ref = (Yr[0], Yr[4], Yr[5] if nvar == 6 else 0.0)
        P = o.primitives(Y, z=z, ref=ref)
        exact = _exact_pressure(cfg, Y, z, nvar) - _exact_pressure(cfg, Yr, z, nvar)
        worst = max(worst, abs(float(Decimal(P["pp"]) - exact)))
        P0 = o.primitives(Yr, z=z, ref=ref)
        assert P0["pp"] == 0.0
    assert worst < 5e-13, worst


def test_flux1_entries(moist):
    """F1 = [rho u; rho u(x)u + p I; (rho e + p) u; rho q u]  (eq. 1, 2, 4, 5)."""
    cfg = moist.cfg
    Y = W.conserved(cfg, np.float64(1.1), 3.0, -2.0, 0.5, np.float64(285.0), np.float64(0.012), np.float64(100.0))
    F = moist.flux1(Y, z=100.0)
    P = moist.primitives(Y, z=100.0)
    u = np.array([P["u"], P["v"], P["w"]])
    assert np.allclose(F[0], Y[1:4], rtol=0, atol=1e-14)
    want = np.outer(Y[1:4], u) + P["p"] * np.eye(3)
    assert np.max(np.abs(F[1:4] - want)) < 1e-9
    assert np.max(np.abs(F[4] - (Y[4] + P["p"]) * u)) < 1e-7
    assert np.max(np.abs(F[5] - Y[5] * u)) < 1e-15


def test_smagorinsky_linear_shear(moist):
    """u = (alpha z, 0, 0): |S| = alpha, nu_t = (C_s Delta)^2 alpha; tau_xz = -nu_t alpha (eq. 33-38)."""
    cfg = moist.cfg
    alpha, J = 0.02, 50.0 * 40.0 * 30.0 / 8
    G = np.zeros((5, 3)); G[0, 2] = alpha
    Y = W.conserved(cfg, np.float64(1.0), 2.0, 1.0, 0.0, np.float64(290.0), np.float64(0.01), np.float64(0.0))
    F2, nu = moist.flux2(Y, G, J)
    Delta = (50.0 * 40.0 * 30.0) ** (1 / 3) / cfg["N"]
    assert abs(nu - (cfg["C_s"] * Delta) ** 2 * alpha) < 1e-12 * nu
    # momentum: rho tau; tau_xz = tau_zx = -2 nu (alpha/2)
    want = np.zeros((3, 3)); want[0, 2] = want[2, 0] = -nu * alpha
    assert np.max(np.abs(F2[1:4] - want)) < 1e-14
    # energy: u . rho tau  (no enthalpy / moisture gradient here)
    assert np.max(np.abs(F2[4] - np.array([0.0, 0.0, -nu * alpha * 2.0]))) < 1e-14
    assert np.max(np.abs(F2[0])) == 0 and np.max(np.abs(F2[5])) == 0


def test_sgs_scalar_fluxes(moist):
    """d_q = -D_t grad q, J + D = -D_t grad h_tot, D_t = nu_t / Pr_t; mass and momentum carry rho d_q (R13)."""
    cfg = moist.cfg
    rng = np.random.default_rng(3)
    G = rng.normal(0, 1e-2, (5, 3)); G[4] *= 1e-3
    J = 125.0
    rho, u = 1.07, np.array([2.0, -1.0, 0.5])
    Y = W.conserved(cfg, np.float64(rho), *u, np.float64(290.0), np.float64(0.01), np.float64(0.0))
    F2, nu = moist.flux2(Y, G, J)
    S = 0.5 * (G[:3] + G[:3].T)
    assert abs(nu - (cfg["C_s"] * (8 * J) ** (1 / 3) / cfg["N"]) ** 2 * np.sqrt(2 * np.sum(S * S))) < 1e-13 * nu
    Dt = nu / cfg["Pr_t"]
    dq = -Dt * G[4]; JD = -Dt * G[3]; tau = -2 * nu * S
    assert np.max(np.abs(F2[0] - rho * dq)) < 1e-16
    assert np.max(np.abs(F2[5] - rho * dq)) < 1e-16
    assert np.max(np.abs(F2[1:4] - (rho * tau + np.outer(Y[1:4], dq)))) < 1e-15
    assert np.max(np.abs(F2[4] - (rho * tau @ u + rho * JD))) < 1e-13


def test_rusanov_consistency_and_symmetry(moist):
    """F*(Y, Y) = n.F1(Y);  F*(Y-, Y+; n) = -F*(Y+, Y-; -n)  (conservation);  eq. (27) with R1."""
    cfg = moist.cfg
    rng = np.random.default_rng(11)
    for _ in range(20):
        n = rng.normal(size=3); n /= np.linalg.norm(n)
        Ym = W.conserved(cfg, np.float64(1.1), *rng.normal(0, 5, 3), np.float64(285.0), np.float64(0.012), np.float64(0.0))
        Yp = W.conserved(cfg, np.float64(1.0), *rng.normal(0, 5, 3), np.float64(295.0), np.float64(0.010), np.float64(0.0))
        F = moist.flux1(Ym)
        assert np.max(np.abs(moist.rusanov(Ym, Ym, n) - F @ n)) < 1e-9
        a = moist.rusanov(Ym, Yp, n); b = moist.rusanov(Yp, Ym, -n)
        assert np.max(np.abs(a + b)) < 1e-9
        # penalty term: F* - average = lambda/2 (Y- - Y+), lambda = max(|u.n| + c)
        Pm, Pp = moist.primitives(Ym), moist.primitives(Yp)
        lam = max(abs(np.dot([Pm["u"], Pm["v"], Pm["w"]], n)) + Pm["c"], abs(np.dot([Pp["u"], Pp["v"], Pp["w"]], n)) + Pp["c"])
        avg = 0.5 * (moist.flux1(Ym) @ n + moist.flux1(Yp) @ n)
        assert np.max(np.abs(a - avg - 0.5 * lam * (Ym - Yp))) < 1e-8


def test_wall_mirror_state_has_no_mass_energy_tracer_flux(moist):
    """(A6)-(A8): Rusanov(Y-, mirror(Y-)) has zero mass, energy and tracer flux; momentum flux is along n."""
    cfg = moist.cfg
    rng = np.random.default_rng(5)
    for _ in range(10):
        n = rng.normal(size=3); n /= np.linalg.norm(n)
        Ym = W.conserved(cfg, np.float64(1.1), *rng.normal(0, 5, 3), np.float64(285.0), np.float64(0.012), np.float64(0.0))
        Yp = Ym.copy(); Yp[1:4] = Ym[1:4] - 2 * np.dot(Ym[1:4], n) * n
        F = moist.rusanov(Ym, Yp, n)
        assert abs(F[0]) < 1e-13 and abs(F[4]) < 1e-7 and abs(F[5]) < 1e-15
        t = F[1:4] - np.dot(F[1:4], n) * n
        assert np.max(np.abs(t)) < 1e-9
