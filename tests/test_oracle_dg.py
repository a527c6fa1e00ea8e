"""Pins for O4, O6, O7, O8, O9, O10 of the oracle at the level of the assembled operator.

Every check compares the oracle with something it did not compute itself: a brute-force dense numpy DG
operator (tests/bruteforce_dg.py), analytic fields, or invariants the method guarantees (free-stream
preservation, discrete conservation P:L593, hydrostatic balance of the reference state P:L77-79,
2.5-D invariance P:L365, weak == strong on LGL nodes, order of accuracy).
"""
import numpy as np
import pytest

import workloads as W
from bruteforce_dg import BruteDG


def noisy_state(cfg, seed, amp=1.0, with_ref=True):
    """Random state with jumps on every face, around a resting hydrostatic-ish column."""
    rng = np.random.default_rng(seed)
    xyz = W.node_coords(cfg)
    z = xyz[..., 2]
    shp = z.shape
    T_r = 300.0 - 0.0065 * z
    rho_r = 1.2 * np.exp(-z / 8000.0)
    q_r = (0.015 - 0.01 * z / 3000.0) if cfg["nvar"] == 6 else np.zeros(shp)
    if with_ref:
        zero = np.zeros(shp)
        Qr = W.conserved(cfg, rho_r, zero, zero, zero, T_r, q_r, z)
        cfg["use_ref"] = 1
        cfg["ref_rho"] = np.ascontiguousarray(Qr[..., 0]); cfg["ref_rhoe"] = np.ascontiguousarray(Qr[..., 4])
        cfg["ref_rhoq"] = np.ascontiguousarray(Qr[..., 5]) if cfg["nvar"] == 6 else None
    rho = rho_r * (1 + 1e-3 * amp * rng.uniform(-1, 1, shp))
    u, v, w = (amp * rng.normal(0, 1, shp) for _ in range(3))
    T = T_r + 0.5 * amp * rng.normal(0, 1, shp)
    q = q_r * (1 + 1e-2 * amp * rng.uniform(-1, 1, shp))
    return W.conserved(cfg, rho, u, v, w, T, q, z)


def relerr(a, b):
    """Per-field max-norm error normalised by the field's max magnitude (reading R19)."""
    return max(np.max(np.abs(a[..., v] - b[..., v])) / np.max(np.abs(b[..., v])) for v in range(a.shape[-1]))


# ------------------------------------------------------------------ brute force
@pytest.mark.parametrize("case", ["periodic_inviscid", "full_dry", "full_moist", "full_moist_N3"])
def test_brute_force(oracle_mod, case):
    if case == "periodic_inviscid":
        cfg = W.base_params(N=2, ne=(2, 2, 2), hi=(40.0, 50.0, 60.0), bc=(0, 0, 0), grav=0.0, sgs=0)
        Q = noisy_state(cfg, 1, with_ref=False)
    elif case == "full_dry":
        cfg = W.base_params(N=2, ne=(2, 2, 2), hi=(40.0, 50.0, 60.0), bc=(0, 1, 1), sgs=1, shf_bottom=80.0)
        Q = noisy_state(cfg, 2)
    elif case == "full_moist":
        cfg = W.base_params(N=2, ne=(2, 2, 2), hi=(40.0, 50.0, 60.0), bc=(0, 0, 1), sgs=1, nvar=6, shf_bottom=50.0)
        Q = noisy_state(cfg, 3)
    else:
        cfg = W.base_params(N=3, ne=(3, 2, 2), hi=(90.0, 50.0, 60.0), bc=(1, 0, 1), sgs=1, nvar=6)
        Q = noisy_state(cfg, 4)
    o = oracle_mod.Oracle(cfg)
    b = BruteDG(cfg)
    if cfg["sgs"]:
        G = o.gradient(Q); Gb = b.gradient(Q)
        for s in range(5 if cfg["nvar"] == 6 else 4):
            assert np.max(np.abs(G[:, :, s] - Gb[:, :, s])) < 1e-11 * np.max(np.abs(Gb[:, :, s])), s
    dQ = o.rhs(Q, "weak"); dQb = b.rhs(Q)
    assert relerr(dQ, dQb) < 1e-11
    assert relerr(o.rhs(Q, "strong"), dQb) < 1e-11


# ------------------------------------------------------------------ weak == strong (R3)
@pytest.mark.parametrize("warped", [False, True])
def test_weak_equals_strong(oracle_mod, warped):
    if warped:
        cfg, _, _ = W.config4(ne=(6, 1, 4), N=4, sgs=1)
        cfg["nvar"] = 5
    else:
        cfg = W.base_params(N=4, ne=(3, 2, 3), hi=(300.0, 200.0, 300.0), bc=(0, 0, 1), sgs=1, nvar=6)
    Q = noisy_state(cfg, 10)
    o = oracle_mod.Oracle(cfg)
    assert relerr(o.rhs(Q, "weak"), o.rhs(Q, "strong")) < 1e-12


# ------------------------------------------------------------------ free-stream preservation
@pytest.mark.parametrize("kind", ["flat", "terrain", "xyz"])
def test_free_stream(oracle_mod, kind):
    if kind == "flat":
        cfg = W.base_params(N=4, ne=(3, 3, 3), hi=(300.0, 200.0, 300.0), bc=(0, 0, 0), grav=0.0, sgs=1, nvar=6)
    elif kind == "terrain":
        cfg, _, _ = W.config4(ne=(8, 1, 4), N=4, sgs=1)
        cfg.update(grav=0.0, use_ref=0, bc=(0, 0, 0))
    else:
        from test_oracle_geometry import _general_cfg
        cfg = _general_cfg(N=3); cfg.update(grav=0.0, bc=(0, 0, 0), sgs=1)
    o = oracle_mod.Oracle(cfg)
    z = o.coords()[..., 2]
    one = np.ones_like(z)
    # the warped meshes are not periodic in z as geometry, but a uniform state has no jumps anyway
    Q = W.conserved(cfg, 1.1 * one, 12.0 * one, -7.0 * one, 3.0 * one, 288.0 * one,
                    (0.01 if cfg["nvar"] == 6 else 0.0) * one, z)
    dx = o.diagnostics(Q)["min_node_dx"]
    for form in ("weak", "strong"):
        dQ = o.rhs(Q, form)
        for v in range(cfg["nvar"]):
            F = np.array([o.flux1(Q[0, 0])[v]]).max()
            Tf = max(abs(F), 1e-300) / dx
            assert np.max(np.abs(dQ[..., v])) < 1e-13 * Tf, (form, v)


# ------------------------------------------------------------------ discrete conservation
@pytest.mark.parametrize("case", ["periodic", "walls_sgs_moist", "terrain_sgs", "shf"])
def test_conservation(oracle_mod, case):
    if case == "periodic":
        cfg = W.base_params(N=4, ne=(3, 2, 2), hi=(300.0, 200.0, 200.0), bc=(0, 0, 0), grav=0.0, sgs=1, nvar=6)
        Q = noisy_state(cfg, 20, with_ref=False)
    elif case == "walls_sgs_moist":
        cfg = W.base_params(N=3, ne=(3, 2, 3), hi=(300.0, 200.0, 300.0), bc=(1, 0, 1), sgs=1, nvar=6)
        Q = noisy_state(cfg, 21)
    elif case == "terrain_sgs":
        cfg, _, _ = W.config4(ne=(6, 1, 4), N=4, sgs=1)
        Q = noisy_state(cfg, 22)
    else:
        cfg = W.base_params(N=4, ne=(3, 2, 2), hi=(300.0, 200.0, 200.0), bc=(0, 0, 1), sgs=1, shf_bottom=120.0)
        Q = noisy_state(cfg, 23)
    o = oracle_mod.Oracle(cfg)
    M = o.mass()
    dQ = o.rhs(Q)
    for v in [0, 4] + ([5] if cfg["nvar"] == 6 else []):
        tot = np.sum(M * dQ[..., v]); ref = np.sum(M * np.abs(dQ[..., v]))
        want = 0.0
        if case == "shf" and v == 4:
            want = 120.0 * 300.0 * 200.0      # SHF * bottom area: energy enters the domain
        assert abs(tot - want) < 1e-12 * ref, (v, tot, ref)
    if cfg["bc"] == (0, 0, 0):   # momentum is conserved too without walls / gravity
        for v in (1, 2, 3):
            assert abs(np.sum(M * dQ[..., v])) < 1e-12 * np.sum(M * np.abs(dQ[..., v]))


def test_conservation_over_steps(oracle_mod):
    """eq. (61)-(62): relative mass and energy change stay at round-off over LSRK54 steps."""
    cfg, Q, dt = W.config2(ne=(6, 1, 4), N=4)
    o = oracle_mod.Oracle(cfg)
    d0 = o.diagnostics(Q)
    Q1 = o.lsrk54(Q, dt, 20)
    d1 = o.diagnostics(Q1)
    assert abs(d1["mass"] - d0["mass"]) < 1e-13 * d0["mass"]
    assert abs(d1["energy"] - d0["energy"]) < 1e-13 * d0["energy"]
    assert np.max(np.abs(Q1 - Q)) > 0


# ------------------------------------------------------------------ hydrostatic balance
@pytest.mark.parametrize("kind", ["bubble_base", "mountain_base", "moist_base"])
def test_reference_state_is_steady(oracle_mod, kind):
    if kind == "bubble_base":
        cfg, Q, dt = W.config2(ne=(4, 1, 6), N=4)
    elif kind == "mountain_base":
        cfg, Q, dt = W.config4(ne=(8, 1, 5), N=4, sgs=1)
    else:
        cfg, Q, dt = W.config5(ne=(2, 2, 6), N=4)
    Qr = np.zeros_like(Q)
    Qr[..., 0] = cfg["ref_rho"]; Qr[..., 4] = cfg["ref_rhoe"]
    if cfg["nvar"] == 6:
        Qr[..., 5] = cfg["ref_rhoq"]
    o = oracle_mod.Oracle(cfg)
    dQ = o.rhs(Qr)
    rho_g = np.max(Qr[..., 0]) * cfg["grav"]
    # momentum: exact zero (p' == 0 bitwise, no flow); scalars: no flux at all
    assert np.max(np.abs(dQ[..., 1:4])) <= 1e-13 * rho_g
    assert np.max(np.abs(dQ[..., 0])) == 0.0 and np.max(np.abs(dQ[..., 4])) <= 1e-13 * rho_g * 300
    # and it stays at rest under forward Euler and LSRK54 (BASELINE invariant)
    assert np.max(np.abs(o.euler(Qr, dt, 5) - Qr)) <= 1e-12 * np.max(np.abs(Qr))
    assert np.max(np.abs(o.lsrk54(Qr, dt, 3)[..., 1:4])) <= 1e-10


def test_hydrostatic_residual_without_reference_converges(oracle_mod):
    """use_ref = 0: the discrete balance grad p = -rho g holds to O(h^N); the residual drops with resolution."""
    res = []
    for nez in (4, 8):
        cfg, Q, dt = W.config2(ne=(2, 1, nez), N=4, sgs=0)
        cfg["hi"] = (cfg["hi"][0], cfg["hi"][1], 8000.0)
        cfg2, Qb, _ = _bubble_base(cfg)
        o = oracle_mod.Oracle(cfg2)
        dQ = o.rhs(Qb)
        res.append(np.max(np.abs(dQ[..., 3])))
    assert res[0] > 0 and res[1] < res[0] / 8.0     # at least 3rd-order decay (N = 4 gives ~16-32x)
    assert res[0] < 1e-3 * 1.2 * 9.81


def _bubble_base(cfg):
    """Unperturbed eq. (41) column on the given mesh, without reference-state subtraction."""
    cfg = dict(cfg); cfg.update(use_ref=0, ref_rho=None, ref_rhoe=None, ref_rhoq=None)
    xyz = W.node_coords(cfg); z = xyz[..., 2]
    cp = cfg["c_vd"] + cfg["R_d"]
    exner = 1.0 - cfg["grav"] * z / (cp * 300.0)
    p = cfg["p_0"] * exner ** (cp / cfg["R_d"])
    T = 300.0 * exner
    rho = p / (cfg["R_d"] * T)
    zero = np.zeros_like(z)
    return cfg, W.conserved(cfg, rho, zero, zero, zero, T, zero, z), None


# ------------------------------------------------------------------ 2.5-D invariance and symmetry
def test_slab_invariance_and_mirror_symmetry(oracle_mod):
    cfg, Q, dt = W.config2(ne=(8, 1, 6), N=4)
    o = oracle_mod.Oracle(cfg)
    Q1 = o.lsrk54(Q, dt, 5)
    dQ = o.rhs(Q1)
    Nq = 5
    # d(rho v)/dt = 0 up to round-off of one flux-derivative term T_f = max|p'| / dx_min (reading R19/R23)
    z = o.coords()[..., 2]
    pp = max(abs(o.primitives(Q1[e, n], z=z[e, n], ref=(cfg["ref_rho"][e, n], cfg["ref_rhoe"][e, n], 0.0))["pp"])
             for e in range(o.Ne) for n in range(0, o.Np, 7))
    assert np.max(np.abs(dQ[..., 2])) <= 1e-11 * pp / o.diagnostics(Q1)["min_node_dx"]
    A = dQ.reshape(6, 1, 8, Nq, Nq, Nq, 5)                                        # [ez, ey, ex, k, j, i, v]
    # y-invariance up to round-off of the Rusanov penalty scale lambda |Y| / dx_min per field
    dg = o.diagnostics(Q1)
    for v in range(5):
        scale = dg["max_wavespeed"] * np.max(np.abs(Q1[..., v])) / dg["min_node_dx"] + np.max(np.abs(dQ[..., v]))
        if v in (1, 2, 3):
            scale += np.max(np.abs(Q1[..., 4])) / dg["min_node_dx"]   # ulp(rho e) enters p' and hence grad p'
        assert np.max(np.abs(A[..., v] - A[:, :, :, :, :1, :, v])) <= 1e-14 * scale, v
    mirror = A[:, :, ::-1, :, :, ::-1].copy()                                     # x -> 2 x_c - x
    mirror[..., 1] *= -1
    for v in (0, 1, 3, 4):      # rho v is identically zero (checked above)
        assert np.max(np.abs(A[..., v] - mirror[..., v])) <= 1e-9 * np.max(np.abs(A[..., v])), v


# ------------------------------------------------------------------ BR1 gradient (O4)
def test_gradient_exact_for_polynomials_flat(oracle_mod):
    cfg = W.base_params(N=3, ne=(3, 3, 3), lo=(-1.0, -1.0, -1.0), hi=(2.0, 1.0, 2.0), bc=(1, 1, 1), grav=0.0, nvar=6)
    o = oracle_mod.Oracle(cfg)
    xyz = o.coords(); x, y, z = xyz[..., 0], xyz[..., 1], xyz[..., 2]
    u = 1 + x * y * z + x ** 3 - 2 * y ** 2 * z
    v = 2 - x ** 2 * y + z ** 3
    w = x * y + y * z ** 2 - 0.5 * x ** 3
    q = 0.01 + 1e-3 * (x * y * z + z ** 3)
    rho = np.ones_like(x); T = 300.0 * np.ones_like(x)
    Q = W.conserved(cfg, rho, u, v, w, T, q, z)
    G = o.gradient(Q)
    e = 13                                             # the centre element: all faces interior
    want = {0: [y * z + 3 * x ** 2, x * z - 4 * y * z, x * y - 2 * y ** 2],
            1: [-2 * x * y, -x ** 2, 3 * z ** 2],
            2: [y - 1.5 * x ** 2, x + z ** 2, 2 * y * z],
            4: [1e-3 * y * z, 1e-3 * x * z, 1e-3 * (x * y + 3 * z ** 2)]}
    for s, g in want.items():
        for c in range(3):
            assert np.max(np.abs(G[e, :, s, c] - g[c][e])) < 1e-12 * max(1.0, np.max(np.abs(g[c][e]))), (s, c)
    # h_tot: with u = 0 and T a polynomial, h = c_pm (T - T_0) + ... is a polynomial of the same degree
    T2 = 300.0 + x ** 3 - y * z
    zero = np.zeros_like(x)
    Q2 = W.conserved(cfg, rho, zero, zero, zero, T2, 0.01 + zero, z)
    G2 = o.gradient(Q2)
    cpm = (cfg["c_vd"] + cfg["R_d"]) * 0.99 + (cfg["c_vv"] + cfg["R_v"]) * 0.01
    for c, g in enumerate([3 * x ** 2, -z, -y]):
        assert np.max(np.abs(G2[e, :, 3, c] - cpm * g[e])) < 1e-13 * 3e5  # h_tot ~ 3e5 J/kg


def test_gradient_linear_field_on_warped_mesh(oracle_mod):
    cfg, _, _ = W.config4(ne=(6, 1, 4), N=4)
    cfg.update(grav=0.0, use_ref=0, bc=(1, 0, 1))
    o = oracle_mod.Oracle(cfg)
    xyz = o.coords(); x, y, z = xyz[..., 0], xyz[..., 1], xyz[..., 2]
    a = np.array([[1e-3, 0.0, -2e-3], [3e-4, 0.0, 5e-4], [-1e-3, 0.0, 2e-3]])
    vel = [5 + a[i, 0] * x + a[i, 2] * z for i in range(3)]
    Q = W.conserved(cfg, np.ones_like(x), *vel, 300.0 + 0 * x, 0 * x, z)
    G = o.gradient(Q)
    Ex, Ey, Ez = cfg["ne"]
    inner = [ex + Ex * ez for ez in range(1, Ez - 1) for ex in range(1, Ex - 1)]
    for i in range(3):
        for c in range(3):
            assert np.max(np.abs(G[inner, :, i, c] - a[i, c])) < 1e-13, (i, c)


def test_gradient_converges_on_taylor_green(oracle_mod):
    """eq. (53)-(54): closed-form grad u of the Taylor-Green field; error drops at order ~N under refinement."""
    errs = []
    for ne in (2, 4):
        cfg = W.base_params(N=4, ne=(ne, ne, ne), lo=(-np.pi,) * 3, hi=(np.pi,) * 3, bc=(0, 0, 0), grav=0.0, sgs=1)
        o = oracle_mod.Oracle(cfg)
        xyz = o.coords(); x, y, z = xyz[..., 0], xyz[..., 1], xyz[..., 2]
        U0 = 100.0
        u = U0 * np.sin(x) * np.cos(y) * np.cos(z); v = -U0 * np.cos(x) * np.sin(y) * np.cos(z)
        Q = W.conserved(cfg, 1.178 + 0 * x, u, v, 0 * x, 300.0 + 0 * x, 0 * x, z)
        G = o.gradient(Q)
        dudx = U0 * np.cos(x) * np.cos(y) * np.cos(z); dudz = -U0 * np.sin(x) * np.cos(y) * np.sin(z)
        dvdy = -U0 * np.cos(x) * np.cos(y) * np.cos(z)
        errs.append(max(np.max(np.abs(G[..., 0, 0] - dudx)), np.max(np.abs(G[..., 0, 2] - dudz)),
                        np.max(np.abs(G[..., 1, 1] - dvdy))))
    assert errs[1] < errs[0] / 10.0 and errs[1] < 0.5


# ------------------------------------------------------------------ inviscid operator on an exact solution
def test_density_wave_convergence(oracle_mod):
    """T_0 = 0, g = 0: rho = 1 + 0.2 sin(2 pi x), u = u0, p = const is an exact Euler solution;
    the DG tendency converges to -u0 d(rho)/dx at order >= N."""
    errs = []
    for ne in (4, 8):
        cfg = W.base_params(N=4, ne=(ne, 1, 1), hi=(1.0, 1.0 / ne, 1.0 / ne), bc=(0, 0, 0), grav=0.0, T_0=0.0)
        o = oracle_mod.Oracle(cfg)
        x = o.coords()[..., 0]
        u0, p0 = 30.0, 1.0e5
        rho = 1 + 0.2 * np.sin(2 * np.pi * x)
        T = p0 / (cfg["R_d"] * rho)
        Q = W.conserved(cfg, rho, u0 + 0 * x, 0 * x, 0 * x, T, 0 * x, 0 * x)
        dQ = o.rhs(Q)
        exact = -u0 * 0.2 * 2 * np.pi * np.cos(2 * np.pi * x)
        errs.append(np.max(np.abs(dQ[..., 0] - exact)))
        assert np.max(np.abs(dQ[..., 1] - u0 * exact)) < 50 * errs[-1] + 1e-6
        assert np.max(np.abs(dQ[..., 4] - 0.5 * u0 ** 2 * exact)) < 1000 * errs[-1] + 1e-6
        assert np.max(np.abs(dQ[..., 2:4])) < 1e-13 * p0 * 2 * ne * ne * 10   # round-off of D applied to the uniform p
    assert errs[1] < errs[0] / 10.0 and errs[1] < 1e-2


# ------------------------------------------------------------------ time stepping (O9)
def test_lsrk54_loop_matches_python_recurrence(oracle_mod):
    cfg, Q, dt = W.config1(ne=(2, 2, 2), N=3)
    o = oracle_mod.Oracle(cfg)
    A, B, C = oracle_mod.lsrk54_coeffs()
    U = Q.copy(); dU = np.zeros_like(U)
    for step in range(2):
        for s in range(5):
            dU = A[s] * dU + dt * o.rhs(U)
            U = U + B[s] * dU
    assert np.max(np.abs(o.lsrk54(Q, dt, 2) - U)) <= 1e-14 * np.max(np.abs(U))
    Ue = Q + dt * o.rhs(Q)
    assert np.max(np.abs(o.euler(Q, dt, 1) - Ue)) == 0.0


def test_lsrk54_is_fourth_order_in_time(oracle_mod):
    cfg, Q, _ = W.config2(ne=(4, 1, 4), N=3, sgs=0)
    o = oracle_mod.Oracle(cfg)
    T = 1.0                                  # stable steps only: dt <= 0.25 s here (limit ~0.4 s)
    ref = o.lsrk54(Q, T / 128, 128)
    e1 = np.max(np.abs(o.lsrk54(Q, T / 4, 4) - ref)[..., 3])
    e2 = np.max(np.abs(o.lsrk54(Q, T / 8, 8) - ref)[..., 3])
    e3 = np.max(np.abs(o.lsrk54(Q, T / 16, 16) - ref)[..., 3])
    assert 13.0 < e1 / e2 < 19.0 and 13.0 < e2 / e3 < 19.0, (e1, e2, e3)


# ------------------------------------------------------------------ sampled evaluation and diagnostics
def test_rhs_elements_equals_full_rhs(oracle_mod):
    cfg, Q, dt = W.config5(ne=(3, 3, 4), N=3)
    o = oracle_mod.Oracle(cfg)
    full = o.rhs(Q)
    el = np.array([0, 7, 17, 35])
    part = o.rhs_elements(Q, el)
    assert np.max(np.abs(part - full[el])) == 0.0
    o2 = oracle_mod.Oracle(cfg, cache_geometry=False)
    assert np.max(np.abs(o2.rhs_elements(Q, el) - full[el])) == 0.0


def test_diagnostics_against_numpy(oracle_mod):
    cfg, Q, dt = W.config5(ne=(2, 2, 3), N=3)
    o = oracle_mod.Oracle(cfg)
    d = o.diagnostics(Q)
    M = o.mass()
    vol = 6000.0 * 2 / 96 * 6000.0 * 2 / 96 * 3000.0
    assert abs(d["volume"] - vol) < 1e-12 * vol
    assert abs(d["mass"] - np.sum(M * Q[..., 0])) < 1e-13 * d["mass"]
    assert abs(d["energy"] - np.sum(M * Q[..., 4])) < 1e-13 * abs(d["energy"])
    assert abs(d["water"] - np.sum(M * Q[..., 5])) < 1e-13 * d["water"]
    u2 = (Q[..., 1:4] ** 2).sum(-1) / Q[..., 0] ** 2
    assert abs(d["kinetic"] - 0.5 * np.sum(M * u2) / vol) < 1e-13 * d["kinetic"]      # eq. (57)
    assert abs(d["max_wavespeed"] - W.sound_speed_max(cfg, Q, W.node_coords(cfg)[..., 2])) < 1e-10
    assert abs(d["min_node_dx"] - W.min_node_spacing(cfg)) < 1e-12 * d["min_node_dx"]
    assert d["n_nonfinite"] == 0
    Q2 = Q.copy(); Q2[0, 0, 0] = np.nan
    assert o.diagnostics(Q2)["n_nonfinite"] == 1
