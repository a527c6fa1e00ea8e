"""Pins for the oracle's saturation adjustment (eq. 15; scope row NEXT-4): temperature and liquid water from
(rho, q_t, I) by Newton iteration with the closed-form saturation vapour pressure of a calorically perfect gas.

What fixes the expected values: the triple point (p* there is p_tr by construction), the Clausius-Clapeyron relation the
closed form integrates (checked by differentiating it in 50-digit arithmetic), states CONSTRUCTED from a chosen temperature
(the oracle has to invert eq. 7-8 back to that temperature), an independent bracketing root finder (scipy brentq on a numpy
restatement of eq. 7-8), continuity at the saturation threshold, and the identities p = rho R_m T, R_m of eq. (14)."""
from decimal import Decimal, getcontext

import numpy as np
import pytest
from scipy.optimize import brentq

import workloads as W

C_VL, P_TR, T_TR, L_V0 = 4181.0, 611.657, 273.16, 2.5008e6     # Table 1 and the triple point of water


def _cfg(**kw):
    c = W.base_params(N=2, ne=(1, 1, 1), hi=(10.0, 10.0, 10.0), nvar=6, grav=9.81, satadj=1)
    c.update(kw)
    return c


def _pvs(c, T):
    dcp = c["c_vv"] + c["R_v"] - C_VL
    return P_TR * (T / T_TR) ** (dcp / c["R_v"]) * np.exp((L_V0 - dcp * c["T_0"]) / c["R_v"] * (1 / T_TR - 1 / T))


def _I_eq(c, T, rho, qt):
    """eq. (7)-(8) at equilibrium (numpy restatement used only to BUILD inputs and for the bracketing root finder)."""
    qvs = _pvs(c, T) / (rho * c["R_v"] * T)
    qv = min(qt, qvs); ql = qt - qv
    return (1 - qt) * c["c_vd"] * (T - c["T_0"]) + qv * (c["c_vv"] * (T - c["T_0"]) + c["I_v0"]) + ql * C_VL * (T - c["T_0"]), ql


def _state(c, rho, T, qt, u=(3.0, -2.0, 0.5), z=7.0):
    I, ql = _I_eq(c, T, rho, qt)
    e = I + 0.5 * sum(x * x for x in u) + c["grav"] * z
    return np.array([rho, rho * u[0], rho * u[1], rho * u[2], rho * e, rho * qt]), ql


def test_saturation_vapour_pressure_closed_form(oracle_mod):
    c = _cfg(); o = oracle_mod.Oracle(c)
    assert abs(o.sat_vapor_pressure(T_TR) - P_TR) <= 1e-13 * P_TR
    # Clausius-Clapeyron: d ln p* / dT = L(T) / (R_v T^2) with L(T) = L_v0 + (c_pv - c_pl)(T - T_0), differentiated in 50 digits
    getcontext().prec = 50
    Rv, dcp, T0 = Decimal(462), Decimal("1397.5") + Decimal(462) - Decimal(4181), Decimal("273.16")
    for T in (255.0, 280.0, 300.0, 315.0):
        Td = Decimal(T)

        def lnp(t):
            return (dcp / Rv) * (t / Decimal("273.16")).ln() + (Decimal("2500800") - dcp * T0) / Rv * (1 / Decimal("273.16") - 1 / t)
        h = Decimal("1e-10")
        dln = (lnp(Td + h) - lnp(Td - h)) / (2 * h)
        L = Decimal("2500800") + dcp * (Td - T0)
        assert abs(dln - L / (Rv * Td * Td)) <= Decimal("1e-18")
        assert abs(o.sat_vapor_pressure(T) - float(Decimal(P_TR) * lnp(Td).exp())) <= 2e-14 * o.sat_vapor_pressure(T)
    # magnitude: 3.5 kPa at 300 K, 1.2 kPa at 283.15 K (steam tables: 3537 Pa, 1228 Pa; constant heat capacities cost < 1 %)
    assert abs(o.sat_vapor_pressure(300.0) / 3537.0 - 1) < 0.01 and abs(o.sat_vapor_pressure(283.15) / 1228.0 - 1) < 0.01


def test_unsaturated_air_is_unchanged(oracle_mod):
    c = _cfg(); o = oracle_mod.Oracle(c); o0 = oracle_mod.Oracle(dict(c, satadj=0))
    Y, ql = _state(c, 1.1, 295.0, 0.010)            # q_v*(295 K, 1.1) ~ 0.0175 > q_t
    assert ql == 0.0
    P, P0 = o.primitives(Y, z=7.0), o0.primitives(Y, z=7.0)
    for k in ("T", "p", "c", "htot", "theta_v"):
        assert P[k] == P0[k], k
    assert P["ql"] == 0.0 and abs(P["T"] - 295.0) <= 1e-12 * 295.0


@pytest.mark.parametrize("rho,T,qt", [(1.1, 295.0, 0.020), (0.95, 282.0, 0.012), (1.2, 300.5, 0.0235), (0.8, 275.0, 0.0075), (1.0, 290.0, 0.0165)])
def test_newton_inverts_the_constructed_state(oracle_mod, rho, T, qt):
    c = _cfg(); o = oracle_mod.Oracle(c)
    Y, ql = _state(c, rho, T, qt)
    assert ql > 0.0                                  # the case really is saturated
    P = o.primitives(Y, z=7.0)
    assert abs(P["T"] - T) <= 1e-12 * T
    assert abs(P["ql"] - ql) <= 1e-12 * qt
    Rm = c["R_d"] * (1 - qt) + c["R_v"] * (qt - ql)                       # eq. (14) with q_c = q_l
    assert abs(P["p"] - rho * Rm * T) <= 1e-12 * P["p"]                   # eq. (13)
    cvm = c["c_vd"] * (1 - qt) + c["c_vv"] * (qt - ql) + C_VL * ql
    assert abs(P["c"] - np.sqrt((1 + Rm / cvm) * Rm * T)) <= 1e-12 * P["c"]
    assert abs(P["htot"] - (Y[4] / rho + Rm * T)) <= 1e-12 * P["htot"]
    # independent bracketing root finder on eq. (15)
    I = Y[4] / rho - 0.5 * (9 + 4 + 0.25) - c["grav"] * 7.0
    Tb = brentq(lambda t: _I_eq(c, t, rho, qt)[0] - I, 200.0, 350.0, xtol=1e-12, rtol=1e-15)
    assert abs(P["T"] - Tb) <= 1e-11 * T


def test_continuity_at_the_saturation_threshold_and_latent_heating(oracle_mod):
    c = _cfg(); o = oracle_mod.Oracle(c); o0 = oracle_mod.Oracle(dict(c, satadj=0))
    rho, T = 1.1, 290.0
    qs = _pvs(c, T) / (rho * c["R_v"] * T)
    Ta, Tb = [o.primitives(_state(c, rho, T, qs * f)[0], z=7.0)["T"] for f in (1 - 1e-9, 1 + 1e-9)]
    assert abs(Ta - Tb) <= 1e-7                      # T is continuous across q_t = q_v*
    # condensation releases latent heat: the adjusted temperature exceeds the no-condensate one by ~ L_v q_l / c_vm
    Y, ql = _state(c, rho, T, 1.3 * qs)
    dT = o.primitives(Y, z=7.0)["T"] - o0.primitives(Y, z=7.0)["T"]
    est = (L_V0 - c["R_v"] * c["T_0"] + (c["c_vv"] - C_VL) * (T - c["T_0"])) * ql / (c["c_vd"] * (1 - 1.3 * qs) + c["c_vv"] * 1.3 * qs)
    assert abs(dT / est - 1) < 0.3 and dT > 1.0           # (q_v* rises with T, so less condenses than at the unadjusted T)


def test_reference_pressure_and_rest_state(oracle_mod):
    # p' = p - p_r with both from the same equation of state: exactly zero at the reference state, and the cloudy resting
    # column stays at rest on the mesh (hydrostatic balance to round-off of p / dx)
    c = _cfg(); o = oracle_mod.Oracle(c)
    Y, ql = _state(c, 1.1, 292.0, 0.019, u=(0, 0, 0))
    P = o.primitives(Y, z=7.0, ref=(Y[0], Y[4], Y[5]))
    assert P["pp"] == 0.0 and P["ql"] > 0
    Yp = Y.copy(); Yp[4] *= 1.0 + 1e-6
    P2 = o.primitives(Yp, z=7.0, ref=(Y[0], Y[4], Y[5]))
    assert abs(P2["pp"] - (o.primitives(Yp, z=7.0)["p"] - o.primitives(Y, z=7.0)["p"])) <= 1e-16 * 1e5
