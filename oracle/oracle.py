"""ctypes front-end of the CPU oracle (oracle/dg_oracle.cpp).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and the cpu_baseline /
``--impl reference`` legs of bench.py.  The product (paper_2110_00853_b200) never imports this and
this module never imports the product.

Oracle data layout: ``Q[e, n, v]`` (lexicographic elements, AoS), see dg_oracle.cpp.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dg_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle_dg.so")


def build(force=False):
    """Compile the oracle with gcc (no fused multiply-add contraction, OpenMP over elements)."""
    if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    cmd = ["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=c++17", _SRC, "-o", _LIB]
    subprocess.check_call(cmd)
    return _LIB


class _Params(C.Structure):
    _fields_ = [
        ("N", C.c_int32), ("ne", C.c_int32 * 3), ("lo", C.c_double * 3), ("hi", C.c_double * 3),
        ("bc", C.c_int32 * 3), ("nvar", C.c_int32), ("geom", C.c_int32),
        ("zsfc_nodes", C.POINTER(C.c_double)), ("xyz", C.POINTER(C.c_double)),
        ("R_d", C.c_double), ("c_vd", C.c_double), ("R_v", C.c_double), ("c_vv", C.c_double),
        ("T_0", C.c_double), ("I_v0", C.c_double), ("grav", C.c_double),
        ("sgs", C.c_int32), ("C_s", C.c_double), ("Pr_t", C.c_double), ("use_ref", C.c_int32),
        ("ref_rho", C.POINTER(C.c_double)), ("ref_rhoe", C.POINTER(C.c_double)), ("ref_rhoq", C.POINTER(C.c_double)),
        ("shf_bottom", C.c_double), ("cache_geometry", C.c_int32),
        ("richardson", C.c_int32), ("p_0", C.c_double),
        ("sponge_alpha", C.c_double), ("sponge_zs", C.c_double), ("sponge_gamma", C.c_int32), ("u_relax", C.c_double * 3),
        ("filter_order", C.c_int32), ("filter_alpha", C.c_double), ("riemann", C.c_int32), ("metric_form", C.c_int32),
        ("drag_cd", C.c_double), ("lhf_bottom", C.c_double), ("evap_bottom", C.c_double),
        ("satadj", C.c_int32), ("c_vl", C.c_double), ("p_tr", C.c_double), ("T_tr", C.c_double),
    ]


_lib = None
_dp = C.POINTER(C.c_double)


def _ptr(a):
    return a.ctypes.data_as(_dp)


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.odg_create.restype = C.c_void_p
        L.odg_create.argtypes = [C.POINTER(_Params)]
        L.odg_destroy.argtypes = [C.c_void_p]
        L.odg_neighbour.restype = C.c_int64
        L.odg_neighbour.argtypes = [C.c_void_p, C.c_int64, C.c_int]
        L.odg_num_threads.restype = C.c_int
        L.odg_sat_vapor_pressure.restype = C.c_double
        L.odg_sat_vapor_pressure.argtypes = [C.c_void_p, C.c_double]
        for name, args in {
            "odg_lgl": [C.c_int, _dp, _dp],
            "odg_dmat": [C.c_int, _dp],
            "odg_lsrk54_coeffs": [_dp, _dp, _dp],
            "odg_coords": [C.c_void_p, _dp],
            "odg_elem_geometry": [C.c_void_p, C.c_int64, _dp, _dp, _dp, _dp, _dp],
            "odg_primitives": [C.c_void_p, _dp, C.c_double, C.c_int, C.c_double, C.c_double, C.c_double, _dp],
            "odg_rusanov": [C.c_void_p, _dp, _dp, _dp, C.c_double, _dp],
            "odg_flux1": [C.c_void_p, _dp, C.c_double, _dp],
            "odg_flux2": [C.c_void_p, _dp, C.c_double, _dp, C.c_double, _dp, _dp, _dp],
            "odg_gradient": [C.c_void_p, _dp, _dp],
            "odg_gradient6": [C.c_void_p, _dp, _dp],
            "odg_elem_dxd": [C.c_void_p, C.c_int64, _dp],
            "odg_lsrk_table": [C.c_void_p, _dp, C.c_double, C.c_int, C.c_int, _dp, _dp],
            "odg_filter": [C.c_void_p, _dp],
            "odg_filter_matrix": [C.c_int, C.c_int, C.c_double, _dp],
            "odg_rhs": [C.c_void_p, _dp, _dp, C.c_int],
            "odg_rhs_elements": [C.c_void_p, _dp, C.POINTER(C.c_int64), C.c_int64, _dp],
            "odg_lsrk54": [C.c_void_p, _dp, C.c_double, C.c_double, C.c_int],
            "odg_euler": [C.c_void_p, _dp, C.c_double, C.c_int],
            "odg_lsrk54_stage": [C.c_void_p, _dp, _dp, C.c_double, C.c_int],
            "odg_diagnostics": [C.c_void_p, _dp, _dp],
            "odg_profiles": [C.c_void_p, _dp, _dp],
        }.items():
            getattr(L, name).argtypes = args
            getattr(L, name).restype = None
        _lib = L
    return _lib


def lgl(N):
    xi = np.zeros(N + 1); w = np.zeros(N + 1)
    lib().odg_lgl(N, _ptr(xi), _ptr(w))
    return xi, w


def dmat(N):
    D = np.zeros((N + 1, N + 1))
    lib().odg_dmat(N, _ptr(D))
    return D


def lsrk54_coeffs():
    A = np.zeros(5); B = np.zeros(5); Cc = np.zeros(5)
    lib().odg_lsrk54_coeffs(_ptr(A), _ptr(B), _ptr(Cc))
    return A, B, Cc


def filter_matrix(N, order, alpha=36.0436533891172):
    F = np.zeros((N + 1, N + 1))
    lib().odg_filter_matrix(N, int(order), float(alpha), _ptr(F))
    return F


def num_threads():
    return lib().odg_num_threads()


class Oracle:
    """One mesh + parameter set.  ``cfg`` is the plain dict produced by workloads.configs (keys = the
    parameter names of SURVEY §8(b))."""

    def __init__(self, cfg, cache_geometry=True):
        L = lib()
        self.cfg = cfg
        self.N = int(cfg["N"]); self.Nq = self.N + 1; self.Np = self.Nq ** 3
        self.ne = tuple(int(v) for v in cfg["ne"])
        self.Ne = self.ne[0] * self.ne[1] * self.ne[2]
        self.nvar = int(cfg.get("nvar", 5))
        p = _Params()
        p.N = self.N
        p.ne[:] = self.ne
        p.lo[:] = [float(v) for v in cfg["lo"]]
        p.hi[:] = [float(v) for v in cfg["hi"]]
        p.bc[:] = [int(v) for v in cfg["bc"]]
        p.nvar = self.nvar
        p.geom = int(cfg.get("geom", 0))
        self._keep = []
        if p.geom == 1:
            z = np.ascontiguousarray(cfg["zsfc_nodes"], dtype=np.float64)
            assert z.size == self.ne[0] * self.Nq * self.ne[1] * self.Nq
            self._keep.append(z); p.zsfc_nodes = _ptr(z)
        if p.geom == 2:
            x = np.ascontiguousarray(cfg["xyz"], dtype=np.float64)
            assert x.size == 3 * self.Ne * self.Np
            self._keep.append(x); p.xyz = _ptr(x)
        for k in ("R_d", "c_vd", "R_v", "c_vv", "T_0", "I_v0", "grav", "C_s", "Pr_t", "shf_bottom"):
            setattr(p, k, float(cfg[k]))
        p.sgs = int(cfg.get("sgs", 0))
        p.use_ref = int(cfg.get("use_ref", 0))
        if p.use_ref:
            for k in ("ref_rho", "ref_rhoe", "ref_rhoq"):
                if cfg.get(k) is None:
                    continue
                a = np.ascontiguousarray(cfg[k], dtype=np.float64)
                assert a.size == self.Ne * self.Np
                self._keep.append(a); setattr(p, k, _ptr(a))
        p.cache_geometry = 1 if cache_geometry else 0
        # optional physics / numerics beyond the five BASELINE configs (defaults = off)
        p.richardson = int(cfg.get("richardson", 0))
        p.p_0 = float(cfg.get("p_0", 1.0e5))
        p.sponge_alpha = float(cfg.get("sponge_alpha", 0.0)); p.sponge_zs = float(cfg.get("sponge_zs", 0.0))
        p.sponge_gamma = int(cfg.get("sponge_gamma", 2))
        p.u_relax[:] = [float(v) for v in cfg.get("u_relax", (0.0, 0.0, 0.0))]
        p.filter_order = int(cfg.get("filter_order", 0)); p.filter_alpha = float(cfg.get("filter_alpha", 36.0436533891172))
        p.riemann = int(cfg.get("riemann", 0)); p.metric_form = int(cfg.get("metric_form", 0))
        p.drag_cd = float(cfg.get("drag_cd", 0.0)); p.lhf_bottom = float(cfg.get("lhf_bottom", 0.0))
        p.evap_bottom = float(cfg.get("evap_bottom", 0.0))
        p.satadj = int(cfg.get("satadj", 0)); p.c_vl = float(cfg.get("c_vl", 0.0))
        p.p_tr = float(cfg.get("p_tr", 0.0)); p.T_tr = float(cfg.get("T_tr", 0.0))
        self._h = L.odg_create(C.byref(p))
        if not self._h:
            raise ValueError("odg_create rejected the parameters")

    def close(self):
        if self._h:
            lib().odg_destroy(self._h); self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- geometry
    def coords(self):
        x = np.zeros((self.Ne, self.Np, 3))
        lib().odg_coords(self._h, _ptr(x))
        return x

    def elem_geometry(self, e):
        Nq, Np = self.Nq, self.Np
        Ja = np.zeros((Np, 3, 3)); J = np.zeros(Np); M = np.zeros(Np)
        sJn = np.zeros((6, Nq, Nq, 3)); lift = np.zeros((6, Nq, Nq))
        lib().odg_elem_geometry(self._h, e, _ptr(Ja), _ptr(J), _ptr(M), _ptr(sJn), _ptr(lift))
        return dict(Ja=Ja, J=J, M=M, sJn=sJn, lift=lift)

    def mass(self):
        M = np.zeros((self.Ne, self.Np))
        for e in range(self.Ne):
            M[e] = self.elem_geometry(e)["M"]
        return M

    def neighbour(self, e, f):
        return int(lib().odg_neighbour(self._h, e, f))

    # ---- pointwise
    def primitives(self, Y, z=0.0, ref=None):
        Y = np.ascontiguousarray(Y, dtype=np.float64); out = np.zeros(12)
        if ref is None:
            lib().odg_primitives(self._h, _ptr(Y), float(z), 0, 0.0, 0.0, 0.0, _ptr(out))
        else:
            lib().odg_primitives(self._h, _ptr(Y), float(z), 1, float(ref[0]), float(ref[1]), float(ref[2]), _ptr(out))
        return dict(zip(("rho", "u", "v", "w", "q", "T", "p", "pp", "htot", "c", "theta_v", "ql"), out))

    def sat_vapor_pressure(self, T):
        return float(lib().odg_sat_vapor_pressure(self._h, float(T)))

    def rusanov(self, Ym, Yp, n, z=0.0):
        Ym = np.ascontiguousarray(Ym, dtype=np.float64); Yp = np.ascontiguousarray(Yp, dtype=np.float64)
        n = np.ascontiguousarray(n, dtype=np.float64); out = np.zeros(self.nvar)
        lib().odg_rusanov(self._h, _ptr(Ym), _ptr(Yp), _ptr(n), float(z), _ptr(out))
        return out

    def flux1(self, Y, z=0.0):
        Y = np.ascontiguousarray(Y, dtype=np.float64); F = np.zeros((self.nvar, 3))
        lib().odg_flux1(self._h, _ptr(Y), float(z), _ptr(F))
        return F

    def flux2(self, Y, G, J, z=0.0, dxd=None):
        """G: [5][3] (u, v, w, h_tot, q) or [6][3] with theta_v; dxd: diagonal of dx/dxi (default: a cube of volume 8 J)."""
        Y = np.ascontiguousarray(Y, dtype=np.float64)
        G6 = np.zeros((6, 3)); G = np.asarray(G, dtype=np.float64); G6[: G.shape[0]] = G
        dxd = np.ascontiguousarray(np.full(3, np.cbrt(J)) if dxd is None else dxd, dtype=np.float64)
        F = np.zeros((self.nvar, 3)); nu = np.zeros(1)
        lib().odg_flux2(self._h, _ptr(Y), float(z), _ptr(G6), float(J), _ptr(dxd), _ptr(F), _ptr(nu))
        return F, float(nu[0])

    def elem_dxd(self, e):
        d = np.zeros((self.Np, 3))
        lib().odg_elem_dxd(self._h, e, _ptr(d))
        return d

    # ---- operators
    def _q(self, Q):
        Q = np.ascontiguousarray(Q, dtype=np.float64)
        assert Q.shape == (self.Ne, self.Np, self.nvar), Q.shape
        return Q

    def gradient(self, Q):
        Q = self._q(Q); G = np.zeros((self.Ne, self.Np, 5, 3))
        lib().odg_gradient(self._h, _ptr(Q), _ptr(G))
        return G

    def gradient6(self, Q):
        Q = self._q(Q); G = np.zeros((self.Ne, self.Np, 6, 3))
        lib().odg_gradient6(self._h, _ptr(Q), _ptr(G))
        return G

    def rhs(self, Q, form="weak"):
        Q = self._q(Q); dQ = np.zeros_like(Q)
        lib().odg_rhs(self._h, _ptr(Q), _ptr(dQ), 0 if form == "weak" else 1)
        return dQ

    def rhs_elements(self, Q, elems):
        Q = self._q(Q); el = np.ascontiguousarray(elems, dtype=np.int64)
        out = np.zeros((el.size, self.Np, self.nvar))
        lib().odg_rhs_elements(self._h, _ptr(Q), el.ctypes.data_as(C.POINTER(C.c_int64)), el.size, _ptr(out))
        return out

    def lsrk54(self, Q, dt, nsteps, t=0.0):
        Q = self._q(Q).copy()
        lib().odg_lsrk54(self._h, _ptr(Q), float(t), float(dt), int(nsteps))
        return Q

    def lsrk_table(self, Q, dt, nsteps, A, B):
        """nsteps steps of the 2N-storage scheme with coefficient tables A, B (A[0] = 0)."""
        Q = self._q(Q).copy()
        A = np.ascontiguousarray(A, dtype=np.float64); B = np.ascontiguousarray(B, dtype=np.float64)
        lib().odg_lsrk_table(self._h, _ptr(Q), float(dt), int(nsteps), int(A.size), _ptr(A), _ptr(B))
        return Q

    def filter(self, Q):
        Q = self._q(Q).copy()
        lib().odg_filter(self._h, _ptr(Q))
        return Q

    def euler(self, Q, dt, nsteps):
        Q = self._q(Q).copy()
        lib().odg_euler(self._h, _ptr(Q), float(dt), int(nsteps))
        return Q

    def lsrk54_stage(self, Q, dU, dt, s):
        """In place on Q and dU (timing helper)."""
        lib().odg_lsrk54_stage(self._h, _ptr(Q), _ptr(dU), float(dt), int(s))

    def diagnostics(self, Q):
        Q = self._q(Q); out = np.zeros(8)
        lib().odg_diagnostics(self._h, _ptr(Q), _ptr(out))
        return dict(zip(("mass", "energy", "water", "kinetic", "max_wavespeed", "min_node_dx", "volume", "n_nonfinite"), out))

    PROFILE_COLUMNS = ("z", "rho") + tuple(f"{p}{v}" for p in ("", "w'", "var_") for v in ("u", "v", "w", "h_tot", "q_t", "theta_v"))

    def profiles(self, Q):
        """Density-weighted horizontal statistics (App. B): array [Ez*Nq][20], columns PROFILE_COLUMNS."""
        Q = self._q(Q); out = np.zeros((self.ne[2] * self.Nq, 20))
        lib().odg_profiles(self._h, _ptr(Q), _ptr(out))
        return out
