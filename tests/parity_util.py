"""Helpers of the GPU parity tests: error norms of reading R19 and small-mesh variants of the five configs."""
import numpy as np

import workloads as W

RHS_TOL = 1e-11     # BASELINE.json north_star: one RHS, max-norm per field / field max magnitude
STEP_TOL = 1e-9     # after 100 LSRK54 steps


def flux_scale(cfg, Q, dx_min):
    """T_f = max|F_f| / dx_min per field (R19): the size of one flux-derivative term."""
    xyz = W.node_coords(cfg)
    z = xyz[..., 2]
    rho = Q[..., 0]
    u = Q[..., 1:4] / rho[..., None]

    def pressure(S):
        r = S[..., 0]
        q = S[..., 5] / r if cfg["nvar"] == 6 else 0.0
        cvm = cfg["c_vd"] * (1 - q) + cfg["c_vv"] * q
        Rm = cfg["R_d"] * (1 - q) + cfg["R_v"] * q
        vel2 = (S[..., 1:4] ** 2).sum(-1) / r ** 2
        T = cfg["T_0"] + (S[..., 4] / r - 0.5 * vel2 - cfg["grav"] * z - q * cfg["I_v0"]) / cvm
        return r * Rm * T

    # full pressure, as in R23: the momentum flux-derivative term is d(p)/dx before the reference is removed
    p = pressure(Q)
    pp = p
    umax = np.abs(u).max()
    T = [np.abs(Q[..., 1:4]).max()]
    for i in range(3):
        T.append(np.abs(Q[..., 1 + i]).max() * umax + np.abs(pp).max())
    T.append((np.abs(Q[..., 4]) + np.abs(p)).max() * umax)
    if cfg["nvar"] == 6:
        T.append(np.abs(Q[..., 5]).max() * umax)
    return np.array(T) / dx_min


def rhs_errors(dQ_gpu, dQ_ora, cfg, Q, dx_min):
    """err_f per field, normalised by max|dQ_ora_f|, or by T_f where the oracle tendency is (numerically) zero."""
    Tf = flux_scale(cfg, Q, dx_min)
    errs = []
    for v in range(dQ_ora.shape[-1]):
        m = np.max(np.abs(dQ_ora[..., v]))
        scale = m if m > 1e-8 * Tf[v] else Tf[v]
        d = np.max(np.abs(dQ_gpu[..., v] - dQ_ora[..., v]))
        errs.append(d / scale if scale > 0 else (0.0 if d == 0 else np.inf))
    return np.array(errs)


def state_errors(Q_gpu, Q_ora):
    """max|Q_gpu - Q_ora| / max|Q_ora| per field; the three momentum components share one scale (in the 2.5-D
    configs rho*v is identically zero up to round-off, R19)."""
    errs = []
    mom = np.max(np.abs(Q_ora[..., 1:4]))
    for v in range(Q_ora.shape[-1]):
        scale = np.max(np.abs(Q_ora[..., v]))
        if v in (1, 2, 3):
            scale = max(scale, mom) if scale < 1e-8 * mom else scale
        errs.append(np.max(np.abs(Q_gpu[..., v] - Q_ora[..., v])) / max(scale, 1e-300))
    return np.array(errs)


def small_config(k, N=4):
    """Meshes the oracle steps in seconds, spanning several CTAs and a ragged last CTA (Ne % EPB != 0)."""
    if k == 1:
        return W.config1(ne=(4, 4, 4), N=N)
    if k == 2:
        return W.config2(ne=(12, 1, 8), N=N)
    if k == 3:
        return W.config3(ne=(5, 4, 6), N=N, hi=(1000.0, 800.0, 1125.0))
    if k == 4:
        return W.config4(ne=(14, 1, 6), N=N)
    if k == 5:
        return W.config5(ne=(6, 5, 7), N=N, hi=(375.0, 312.5, 3000.0))
    raise ValueError(k)
