"""Seeded synthetic inputs shaped like the paper's cases (BASELINE.json configs 1-5).

This module serves BOTH the oracle tests and the CUDA path (tests, bench.py).  It holds no DG
arithmetic: it only lays out node coordinates of a brick mesh, evaluates analytic/tabulated
atmospheric profiles, draws seeded random perturbations, and converts (rho, u, T, q) to the
conserved state.  It imports neither ``oracle`` nor ``paper_2110_00853_b200``.

Shapes stand in for the paper's benchmarks (P:L<n> = PAPER.md line):
  config 2  rising thermal bubble, eq. (41), bubble shape reading R15
  config 3  dry convective boundary layer box (stable layer above a mixed layer, surface heat flux)
  config 4  flow over a bell-shaped mountain, eq. (49)-(51) P:L453-466 (reading R17 for eq. 51)
  config 5  moist shallow-cumulus-shaped box (layering described at P:L553; round synthetic numbers;
            the BOMEX case tables themselves are not reproduced)
All arrays are lexicographic: element e = ex + Ex*(ey + Ey*ez), node n = i + Nq*(j + Nq*k),
state Q[e, n, v] with v = rho, rho*u, rho*v, rho*w, rho*e_tot, [rho*q_tot].
"""
import numpy as np

SEED0 = 211000853

TABLE1 = dict(R_d=287.0, R_v=462.0, c_vd=717.5, c_vv=1397.5, T_0=273.16, L_v0=2.5008e6)


def lgl_nodes(N):
    """Legendre-Gauss-Lobatto points on [-1, 1] from numpy's Legendre class (library routine)."""
    from numpy.polynomial import legendre as L
    c = np.zeros(N + 1); c[N] = 1.0
    dc = L.legder(c)
    x = np.sort(np.real(L.legroots(dc))) if N > 1 else np.array([])
    ddc = L.legder(dc)
    for _ in range(3):  # Newton polish
        x = x - L.legval(x, dc) / L.legval(x, ddc) if x.size else x
    x = 0.5 * (x - x[::-1]) if x.size else x
    return np.concatenate([[-1.0], x, [1.0]])


def base_params(**kw):
    p = dict(N=4, ne=(4, 4, 4), lo=(0.0, 0.0, 0.0), hi=(1.0, 1.0, 1.0), bc=(0, 0, 0), nvar=5, geom=0,
             zsfc_nodes=None, xyz=None, R_d=TABLE1["R_d"], c_vd=TABLE1["c_vd"], R_v=TABLE1["R_v"],
             c_vv=TABLE1["c_vv"], T_0=TABLE1["T_0"], I_v0=TABLE1["L_v0"] - TABLE1["R_v"] * TABLE1["T_0"],
             grav=9.81, sgs=0, C_s=0.21, Pr_t=1.0 / 3.0, use_ref=0, ref_rho=None, ref_rhoe=None,
             ref_rhoq=None, shf_bottom=0.0, p_0=1.0e5)
    p.update(kw)
    return p


def node_coords(cfg):
    """xyz[e, n, 3] of the brick mesh (with the linear-decay terrain warp if geom == 1)."""
    N = cfg["N"]; Nq = N + 1
    Ex, Ey, Ez = cfg["ne"]
    xi = lgl_nodes(N)
    ax = []
    for d, E in enumerate((Ex, Ey, Ez)):
        h = (cfg["hi"][d] - cfg["lo"][d]) / E
        ax.append(cfg["lo"][d] + (np.arange(E)[:, None] + 0.5 * (xi[None, :] + 1.0)) * h)  # [E, Nq]
    X = np.broadcast_to(ax[0][None, None, :, None, None, :], (Ez, Ey, Ex, Nq, Nq, Nq))
    Y = np.broadcast_to(ax[1][None, :, None, None, :, None], (Ez, Ey, Ex, Nq, Nq, Nq))
    Z = np.broadcast_to(ax[2][:, None, None, :, None, None], (Ez, Ey, Ex, Nq, Nq, Nq))
    xyz = np.stack([X, Y, Z], axis=-1).reshape(Ex * Ey * Ez, Nq ** 3, 3).copy()
    if cfg.get("geom", 0) == 1:
        zs = np.asarray(cfg["zsfc_nodes"]).reshape(Ey, Nq, Ex, Nq)            # [ey, j, ex, i]
        zs = np.broadcast_to(zs.transpose(0, 2, 1, 3)[None, :, :, None, :, :], (Ez, Ey, Ex, Nq, Nq, Nq))
        zs = zs.reshape(Ex * Ey * Ez, Nq ** 3)
        zt = xyz[:, :, 2]
        xyz[:, :, 2] = zt + zs * (cfg["hi"][2] - zt) / (cfg["hi"][2] - cfg["lo"][2])
    return xyz


def min_node_spacing(cfg):
    xi = lgl_nodes(cfg["N"])
    return min((cfg["hi"][d] - cfg["lo"][d]) / cfg["ne"][d] for d in range(3)) * 0.5 * (xi[1] - xi[0])


# ------------------------------------------------------------------ thermodynamic conversions (inputs only)
def _mix(cfg, q):
    cvm = cfg["c_vd"] * (1.0 - q) + cfg["c_vv"] * q
    Rm = cfg["R_d"] * (1.0 - q) + cfg["R_v"] * q
    return cvm, Rm


def conserved(cfg, rho, u, v, w, T, q, z):
    """(rho, velocity, T, q_t, height) -> Q[..., nvar]  (eq. 6-10 with q_l = q_i = 0)."""
    cvm, _ = _mix(cfg, q)
    e = cvm * (T - cfg["T_0"]) + q * cfg["I_v0"] + 0.5 * (u * u + v * v + w * w) + cfg["grav"] * z
    fields = [rho, rho * u, rho * v, rho * w, rho * e]
    if cfg["nvar"] == 6:
        fields.append(rho * q)
    return np.stack(fields, axis=-1)


def sound_speed_max(cfg, Q, z):
    rho = Q[..., 0]
    u = Q[..., 1:4] / rho[..., None]
    q = Q[..., 5] / rho if cfg["nvar"] == 6 else 0.0
    cvm, Rm = _mix(cfg, q)
    eint = Q[..., 4] / rho - 0.5 * (u ** 2).sum(-1) - cfg["grav"] * z
    T = cfg["T_0"] + (eint - q * cfg["I_v0"]) / cvm
    c = np.sqrt((1.0 + Rm / cvm) * Rm * T)
    return float((np.sqrt((u ** 2).sum(-1)) + c).max())


def _theta_to_state(cfg, theta, p, q):
    cvm, Rm = _mix(cfg, q)
    T = theta * (p / cfg["p_0"]) ** (Rm / (cvm + Rm))
    rho = p / (Rm * T)
    return rho, T


def _attach_ref(cfg, rho_r, T_r, q_r, z):
    cfg = dict(cfg)
    zero = np.zeros_like(rho_r)
    Qr = conserved(cfg, rho_r, zero, zero, zero, T_r, q_r, z)
    cfg["use_ref"] = 1
    cfg["ref_rho"] = np.ascontiguousarray(Qr[..., 0])
    cfg["ref_rhoe"] = np.ascontiguousarray(Qr[..., 4])
    cfg["ref_rhoq"] = np.ascontiguousarray(Qr[..., 5]) if cfg["nvar"] == 6 else None
    return cfg


# ------------------------------------------------------------------ the five configurations
def config1(ne=(4, 4, 4), N=4, seed=SEED0 + 1, nvar=5):
    """Triply periodic box, i.i.d. noisy state (every face carries jumps), g = 0, inviscid."""
    L = 1000.0 * np.array(ne) / 4.0
    cfg = base_params(N=N, ne=tuple(ne), hi=tuple(L), bc=(0, 0, 0), nvar=nvar, c_vd=717.0, grav=0.0, sgs=0)
    xyz = node_coords(cfg)
    rng = np.random.default_rng(seed)
    shp = xyz.shape[:2]
    rho = 1.2 + 1e-3 * rng.uniform(-1, 1, shp)
    u, v, w = (rng.normal(0, 1, shp) for _ in range(3))
    T = 300.0 + 0.1 * rng.normal(0, 1, shp)
    q = 0.01 + 1e-4 * rng.uniform(-1, 1, shp) if nvar == 6 else np.zeros(shp)
    Q = conserved(cfg, rho, u, v, w, T, q, xyz[..., 2])
    dt = 1e-3 * min_node_spacing(cfg) / sound_speed_max(cfg, Q, xyz[..., 2])
    return cfg, Q, dt


def _bubble_profile(cfg, z, theta0=300.0):
    cp = cfg["c_vd"] + cfg["R_d"]
    exner = 1.0 - cfg["grav"] * z / (cp * theta0)               # eq. (41)
    p = cfg["p_0"] * exner ** (cp / cfg["R_d"])
    return p


def config2(ne=(40, 1, 20), N=4, sgs=1, seed=SEED0 + 2):
    """2.5-D rising thermal bubble: theta_0 = 300 K, cos^2 bubble of 2 K (R15)."""
    Ex, Ey, Ez = ne
    cfg = base_params(N=N, ne=tuple(ne), hi=(500.0 * Ex, 500.0 * Ey, 500.0 * Ez), bc=(0, 0, 1), sgs=sgs)
    xyz = node_coords(cfg)
    x, z = xyz[..., 0], xyz[..., 2]
    p = _bubble_profile(cfg, z)
    zero = np.zeros_like(z)
    rho_r, T_r = _theta_to_state(cfg, 300.0 + zero, p, zero)
    cfg = _attach_ref(cfg, rho_r, T_r, zero, z)
    xc, zc, r0 = 0.5 * cfg["hi"][0], 2000.0, 2000.0
    r = np.sqrt((x - xc) ** 2 + (z - zc) ** 2)
    dth = np.where(r <= r0, 2.0 * np.cos(0.5 * np.pi * r / r0) ** 2, 0.0)
    rho, T = _theta_to_state(cfg, 300.0 + dth, p, zero)
    Q = conserved(cfg, rho, zero, zero, zero, T, zero, z)
    dt = 0.4 * min_node_spacing(cfg) / sound_speed_max(cfg, Q, z)
    return cfg, Q, dt


def config3(ne=(32, 32, 16), N=4, seed=SEED0 + 3, hi=None):
    """Dry convective-boundary-layer box: mixed layer to 1 km, +3 K/km above, noise below 400 m, SHF."""
    Ex, Ey, Ez = ne
    if hi is None:
        hi = (200.0 * Ex, 200.0 * Ey, 187.5 * Ez)
    cfg = base_params(N=N, ne=tuple(ne), hi=tuple(hi), bc=(0, 0, 1), sgs=1, shf_bottom=100.0)
    xyz = node_coords(cfg)
    z = xyz[..., 2]
    cp = cfg["c_vd"] + cfg["R_d"]; g = cfg["grav"]; th0 = 300.0; gam = 0.003; z1 = 1000.0
    theta = np.where(z <= z1, th0, th0 + gam * (z - z1))
    ex1 = 1.0 - g * z1 / (cp * th0)
    exner = np.where(z <= z1, 1.0 - g * z / (cp * th0), ex1 - g / (cp * gam) * np.log(theta / th0))
    p = cfg["p_0"] * exner ** (cp / cfg["R_d"])
    zero = np.zeros_like(z)
    rho_r, T_r = _theta_to_state(cfg, theta, p, zero)
    cfg = _attach_ref(cfg, rho_r, T_r, zero, z)
    rng = np.random.default_rng(seed)
    dth = np.where(z < 400.0, 0.1 * rng.uniform(-1, 1, z.shape), 0.0)
    rho, T = _theta_to_state(cfg, theta + dth, p, zero)
    Q = conserved(cfg, rho, zero, zero, zero, T, zero, z)
    dt = 0.4 * min_node_spacing(cfg) / sound_speed_max(cfg, Q, z)
    return cfg, Q, dt


def config4(ne=(120, 1, 30), N=4, sgs=0, seed=SEED0 + 4):
    """Uniform 10 m/s flow over a bell-shaped mountain on a terrain-following mesh (eq. 49-51)."""
    Ex, Ey, Ez = ne
    cfg = base_params(N=N, ne=tuple(ne), hi=(2500.0 * Ex, 2500.0 * Ey, 700.0 * Ez), bc=(0, 0, 1), sgs=sgs, geom=1)
    Nq = N + 1
    xi = lgl_nodes(N)
    hx = cfg["hi"][0] / Ex
    xb = ((np.arange(Ex)[:, None] + 0.5 * (xi[None, :] + 1.0)) * hx).reshape(-1)        # [Ex*Nq]
    hm, a, xc = 250.0, 5000.0, 0.5 * cfg["hi"][0]
    zs1 = hm * a * a / ((xb - xc) ** 2 + a * a)                                         # eq. (49)
    cfg["zsfc_nodes"] = np.ascontiguousarray(np.broadcast_to(zs1[None, :], (Ey * Nq, Ex * Nq)))
    xyz = node_coords(cfg)
    z = xyz[..., 2]
    g = cfg["grav"]; cp = cfg["c_vd"] + cfg["R_d"]; Nbv = 0.01; th_s = 280.0; p_s = cfg["p_0"]
    theta = th_s * np.exp(Nbv ** 2 * z / g)
    p = p_s * (1.0 + g * g / (cp * th_s * Nbv ** 2) * (np.exp(-Nbv ** 2 * z / g) - 1.0)) ** (cp / cfg["R_d"])   # eq. (50)
    rho = p_s * (p / p_s) ** (cfg["c_vd"] / cp) / (cfg["R_d"] * theta)                  # eq. (51) as corrected by R17
    T = p / (cfg["R_d"] * rho)
    zero = np.zeros_like(z)
    cfg = _attach_ref(cfg, rho, T, zero, z)
    Q = conserved(cfg, rho, 10.0 + zero, zero, zero, T, zero, z)
    dt = 0.4 * min_node_spacing(cfg) / sound_speed_max(cfg, Q, z)
    return cfg, Q, dt


def _moist_column(cfg, heights):
    """Hydrostatic p at the given heights: dp/dz = -rho g by RK4 with 1 m sub-steps from p_0 at z = 0."""
    g = cfg["grav"]

    def theta_of(z):
        return np.where(z <= 500.0, 299.0,
               np.where(z <= 1500.0, 299.0 + 0.004 * (z - 500.0),
               np.where(z <= 2000.0, 303.0 + 0.007 * (z - 1500.0), 306.5 + 0.003 * (z - 2000.0))))

    def q_of(z):
        return 0.017 - 0.013 * z / 3000.0

    def rhs(z, p):
        rho, _ = _theta_to_state(cfg, theta_of(z), p, q_of(z))
        return -rho * g

    def rk4(z, p, h):
        k1 = rhs(z, p); k2 = rhs(z + 0.5 * h, p + 0.5 * h * k1)
        k3 = rhs(z + 0.5 * h, p + 0.5 * h * k2); k4 = rhs(z + h, p + h * k3)
        return p + h / 6.0 * (k1 + 2 * k2 + 2 * k3 + k4)

    zmax = float(np.max(heights))
    nz = int(np.floor(zmax)) + 1
    pg = np.empty(nz + 1); pg[0] = cfg["p_0"]
    for m in range(nz):
        pg[m + 1] = rk4(float(m), pg[m], 1.0)
    base = np.floor(heights).astype(np.int64)
    p = rk4(base.astype(np.float64), pg[base], heights - base)
    return p, theta_of(heights), q_of(heights)


def config5(ne=(96, 96, 48), N=4, seed=SEED0 + 5, hi=None):
    """Moist shallow-cumulus-shaped box: 6 prognostics, conditionally unstable theta, q_t 17 -> 4 g/kg."""
    Ex, Ey, Ez = ne
    if hi is None:
        hi = (6000.0 * Ex / 96.0, 6000.0 * Ey / 96.0, 3000.0)
    cfg = base_params(N=N, ne=tuple(ne), hi=tuple(hi), bc=(0, 0, 1), nvar=6, sgs=1)
    Nq = N + 1
    xi = lgl_nodes(N)
    hz = cfg["hi"][2] / Ez
    zcol = ((np.arange(Ez)[:, None] + 0.5 * (xi[None, :] + 1.0)) * hz)                   # [Ez, Nq]
    p_c, th_c, q_c = _moist_column(cfg, zcol.reshape(-1))
    rho_c, T_c = _theta_to_state(cfg, th_c, p_c, q_c)
    nh = Ex * Ey

    def spread(col):  # [Ez*Nq] -> [Ne, Np] (depends on ez and k only)
        a = col.reshape(Ez, 1, Nq, 1)
        return np.broadcast_to(a, (Ez, nh, Nq, Nq * Nq)).reshape(Ez * nh, Nq ** 3)

    z = spread(zcol.reshape(-1))
    cfg = _attach_ref(cfg, spread(rho_c), spread(T_c), spread(q_c), z)
    rng = np.random.default_rng(seed)
    shp = z.shape
    low = z < 1600.0
    theta = spread(th_c) + np.where(low, 0.1 * rng.uniform(-1, 1, shp), 0.0)
    q = spread(q_c) + np.where(low, 2.5e-5 * rng.uniform(-1, 1, shp), 0.0)
    rho, T = _theta_to_state(cfg, theta, spread(p_c), q)
    u, v, w = (rng.normal(0, 0.1, shp) for _ in range(3))
    Q = conserved(cfg, rho, u, v, w, T, q, z)
    dt = 0.4 * min_node_spacing(cfg) / sound_speed_max(cfg, Q, z)
    return cfg, Q, dt


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}

# element counts of the fixed-DOF sweep of config 5 (SURVEY §8 sizes table)
SWEEP5 = {3: (120, 120, 60), 4: (96, 96, 48), 5: (80, 80, 40), 6: (68, 68, 35)}
