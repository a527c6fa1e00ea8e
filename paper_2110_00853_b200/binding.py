"""ctypes binding of include/cm_dg.h: argument marshalling only, every step of the path runs in the CUDA
library.  Function names equal the C entry points; ``CmDg`` is a small convenience wrapper around a ctx."""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBPATH = os.path.join(_HERE, "libcm_dg.so")


class CmDgError(RuntimeError):
    pass


class _Params(C.Structure):
    _fields_ = [
        ("N", C.c_int32), ("ne", C.c_int32 * 3), ("lo", C.c_double * 3), ("hi", C.c_double * 3),
        ("bc", C.c_int32 * 3), ("nvar", C.c_int32), ("geom", C.c_int32),
        ("zsfc_nodes", C.c_void_p), ("xyz", C.c_void_p),
        ("R_d", C.c_double), ("c_vd", C.c_double), ("R_v", C.c_double), ("c_vv", C.c_double),
        ("T_0", C.c_double), ("I_v0", C.c_double), ("grav", C.c_double),
        ("sgs", C.c_int32), ("C_s", C.c_double), ("Pr_t", C.c_double), ("use_ref", C.c_int32),
        ("ref_rho", C.c_void_p), ("ref_rhoe", C.c_void_p), ("ref_rhoq", C.c_void_p),
        ("shf_bottom", C.c_double),
        ("richardson", C.c_int32), ("p_0", C.c_double),
        ("sponge_alpha", C.c_double), ("sponge_zs", C.c_double), ("sponge_gamma", C.c_int32), ("u_relax", C.c_double * 3),
        ("filter_order", C.c_int32), ("filter_alpha", C.c_double), ("riemann", C.c_int32), ("metric_form", C.c_int32),
        ("drag_cd", C.c_double), ("lhf_bottom", C.c_double), ("evap_bottom", C.c_double),
        ("satadj", C.c_int32), ("c_vl", C.c_double), ("p_triple", C.c_double), ("T_triple", C.c_double),
    ]


class _Tuning(C.Structure):
    _fields_ = [("order_lex", C.c_int32), ("max_chunk", C.c_int32), ("max_patch", C.c_int32), ("force_general", C.c_int32),
                ("kernel", C.c_int32), ("ahead_t", C.c_int32), ("ahead_g", C.c_int32), ("row_len", C.c_int32),
                ("no_graph", C.c_int32), ("no_terrain", C.c_int32)]


class _Diag(C.Structure):
    _fields_ = [("mass", C.c_double), ("energy", C.c_double), ("water", C.c_double), ("kinetic", C.c_double),
                ("max_wavespeed", C.c_double), ("min_node_dx", C.c_double), ("volume", C.c_double),
                ("n_nonfinite", C.c_int64)]


class _StaticDesc(C.Structure):
    _fields_ = [("N", C.c_int32), ("nvar", C.c_int32), ("n_elem", C.c_int64), ("field_stride", C.c_int64),
                ("R_d", C.c_double), ("c_vd", C.c_double), ("R_v", C.c_double), ("c_vv", C.c_double),
                ("T_0", C.c_double), ("I_v0", C.c_double), ("grav", C.c_double)]


class _KStats(C.Structure):
    _fields_ = [("launches_gradient", C.c_int64), ("launches_tendency", C.c_int64), ("launches_other", C.c_int64),
                ("ms_gradient", C.c_double), ("ms_tendency", C.c_double), ("ms_other", C.c_double)]


EXPORTS = ("cm_dg_setup", "cm_dg_setup_tuned", "cm_dg_layout", "cm_dg_coords", "cm_dg_metrics", "cm_dg_gradient", "cm_dg_rhs",
           "cm_dg_lsrk_step", "cm_dg_lsrk_step_table", "cm_dg_filter", "cm_dg_diagnostics", "cm_dg_diagnostics_static", "cm_dg_profiles", "cm_dg_rhs_host", "cm_dg_lsrk_step_host",
           "cm_dg_profile_begin", "cm_dg_profile_end", "cm_dg_destroy", "cm_dg_last_error")

_lib = None


def library_path():
    return _LIBPATH


def _load():
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIBPATH):
        raise CmDgError("CUDA library %s is missing: build it with `python -m paper_2110_00853_b200.build` "
                        "(there is no CPU fallback)" % _LIBPATH)
    L = C.CDLL(_LIBPATH)
    vp, dbl, i32, i64 = C.c_void_p, C.c_double, C.c_int32, C.c_int64
    L.cm_dg_setup.argtypes = [C.POINTER(_Params), vp, C.POINTER(vp)]
    L.cm_dg_setup_tuned.argtypes = [C.POINTER(_Params), C.POINTER(_Tuning), vp, C.POINTER(vp)]
    L.cm_dg_layout.argtypes = [vp, C.POINTER(i64), C.POINTER(i32), C.POINTER(i64), vp]
    L.cm_dg_coords.argtypes = [vp, vp]
    L.cm_dg_metrics.argtypes = [vp, vp, vp]
    L.cm_dg_gradient.argtypes = [vp, vp, vp]
    L.cm_dg_rhs.argtypes = [vp, vp, vp, dbl]
    L.cm_dg_lsrk_step.argtypes = [vp, vp, dbl, dbl, i32]
    L.cm_dg_lsrk_step_table.argtypes = [vp, vp, dbl, dbl, i32, i32, vp, vp, vp]
    L.cm_dg_filter.argtypes = [vp, vp]
    L.cm_dg_diagnostics.argtypes = [vp, vp, C.POINTER(_Diag)]
    L.cm_dg_diagnostics_static.argtypes = [C.POINTER(_StaticDesc), vp, vp, vp, vp, C.POINTER(_Diag)]
    L.cm_dg_profiles.argtypes = [vp, vp, vp, i32]
    L.cm_dg_rhs_host.argtypes = [vp, vp, vp, dbl]
    L.cm_dg_lsrk_step_host.argtypes = [vp, vp, dbl, dbl, i32]
    L.cm_dg_profile_begin.argtypes = [vp]
    L.cm_dg_profile_end.argtypes = [vp, C.POINTER(_KStats)]
    L.cm_dg_destroy.argtypes = [vp]
    L.cm_dg_destroy.restype = None
    L.cm_dg_last_error.restype = C.c_char_p
    for n in EXPORTS:
        if n not in ("cm_dg_destroy", "cm_dg_last_error"):
            getattr(L, n).restype = C.c_int
    _lib = L
    return L


def cm_dg_last_error():
    return _load().cm_dg_last_error().decode()


def _check(rc, what):
    if rc != 0:
        raise CmDgError("%s failed (%d): %s" % (what, rc, cm_dg_last_error()))


def _dptr(t):
    """Device pointer of a torch CUDA tensor (or a raw int)."""
    if isinstance(t, int):
        return C.c_void_p(t)
    assert t.is_cuda and t.is_contiguous() and t.dtype.is_floating_point and t.element_size() == 8
    return C.c_void_p(t.data_ptr())


def _hptr(a):
    """Host pointer of a numpy array or a CPU torch tensor (float64, contiguous)."""
    if isinstance(a, np.ndarray):
        assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
        return C.c_void_p(a.ctypes.data)
    assert (not a.is_cuda) and a.is_contiguous() and a.element_size() == 8
    return C.c_void_p(a.data_ptr())


def cm_dg_setup(cfg, stream=None, tuning=None):
    """cfg: dict with the fields of cm_dg_params (numpy arrays for the HOST pointers); tuning: dict with fields of
    cm_dg_tuning (cm_dg_setup_tuned) or None (cm_dg_setup).  Returns the ctx handle."""
    L = _load()
    p = _Params()
    p.N = int(cfg["N"])
    p.ne[:] = [int(v) for v in cfg["ne"]]
    p.lo[:] = [float(v) for v in cfg["lo"]]
    p.hi[:] = [float(v) for v in cfg["hi"]]
    p.bc[:] = [int(v) for v in cfg["bc"]]
    p.nvar = int(cfg.get("nvar", 5))
    p.geom = int(cfg.get("geom", 0))
    keep = []

    def host(key):
        a = cfg.get(key)
        if a is None:
            return None
        a = np.ascontiguousarray(a, dtype=np.float64)
        keep.append(a)
        return C.c_void_p(a.ctypes.data)

    if p.geom == 1:
        p.zsfc_nodes = host("zsfc_nodes")
    if p.geom == 2:
        p.xyz = host("xyz")
    for k in ("R_d", "c_vd", "R_v", "c_vv", "T_0", "I_v0", "grav", "C_s", "Pr_t", "shf_bottom"):
        setattr(p, k, float(cfg[k]))
    p.sgs = int(cfg.get("sgs", 0))
    for k in ("richardson", "sponge_gamma", "filter_order", "riemann", "metric_form", "satadj"):
        setattr(p, k, int(cfg.get(k, 0)))
    for k in ("p_0", "sponge_alpha", "sponge_zs", "filter_alpha", "drag_cd", "lhf_bottom", "evap_bottom", "c_vl"):
        setattr(p, k, float(cfg.get(k, 0.0)))
    p.u_relax[:] = [float(v) for v in cfg.get("u_relax", (0.0, 0.0, 0.0))]
    p.p_triple = float(cfg.get("p_tr", 0.0)); p.T_triple = float(cfg.get("T_tr", 0.0))
    p.use_ref = int(cfg.get("use_ref", 0))
    if p.use_ref:
        p.ref_rho = host("ref_rho"); p.ref_rhoe = host("ref_rhoe"); p.ref_rhoq = host("ref_rhoq")
    ctx = C.c_void_p()
    sp = C.c_void_p(int(stream.cuda_stream)) if stream is not None else C.c_void_p(0)
    if tuning is None:
        _check(L.cm_dg_setup(C.byref(p), sp, C.byref(ctx)), "cm_dg_setup")
    else:
        tn = _Tuning(ahead_t=-1, ahead_g=-1)
        for k, v in tuning.items():
            if k not in dict(_Tuning._fields_):
                raise CmDgError("unknown tuning field %r" % k)
            setattr(tn, k, int(v))
        _check(L.cm_dg_setup_tuned(C.byref(p), C.byref(tn), sp, C.byref(ctx)), "cm_dg_setup_tuned")
    return ctx


def cm_dg_layout(ctx):
    L = _load()
    ne, npn, st = C.c_int64(), C.c_int32(), C.c_int64()
    _check(L.cm_dg_layout(ctx, C.byref(ne), C.byref(npn), C.byref(st), None), "cm_dg_layout")
    lex = np.zeros(ne.value, dtype=np.int32)
    _check(L.cm_dg_layout(ctx, None, None, None, C.c_void_p(lex.ctypes.data)), "cm_dg_layout")
    return ne.value, npn.value, st.value, lex


def cm_dg_coords(ctx, xyz_dev):
    _check(_load().cm_dg_coords(ctx, _dptr(xyz_dev)), "cm_dg_coords")


def cm_dg_metrics(ctx, Ja_dev, J_dev):
    _check(_load().cm_dg_metrics(ctx, _dptr(Ja_dev), _dptr(J_dev)), "cm_dg_metrics")


def cm_dg_gradient(ctx, Q_dev, G_dev):
    _check(_load().cm_dg_gradient(ctx, _dptr(Q_dev), _dptr(G_dev)), "cm_dg_gradient")


def cm_dg_rhs(ctx, Q_dev, dQ_dev, t=0.0):
    _check(_load().cm_dg_rhs(ctx, _dptr(Q_dev), _dptr(dQ_dev), float(t)), "cm_dg_rhs")


def cm_dg_lsrk_step(ctx, Q_dev, t, dt, nsteps):
    _check(_load().cm_dg_lsrk_step(ctx, _dptr(Q_dev), float(t), float(dt), int(nsteps)), "cm_dg_lsrk_step")


def cm_dg_lsrk_step_table(ctx, Q_dev, t, dt, nsteps, A, B, Cc=None):
    A = np.ascontiguousarray(A, dtype=np.float64); B = np.ascontiguousarray(B, dtype=np.float64)
    assert A.size == B.size
    cp = C.c_void_p(np.ascontiguousarray(Cc, dtype=np.float64).ctypes.data) if Cc is not None else C.c_void_p(0)
    _check(_load().cm_dg_lsrk_step_table(ctx, _dptr(Q_dev), float(t), float(dt), int(nsteps), int(A.size),
                                         C.c_void_p(A.ctypes.data), C.c_void_p(B.ctypes.data), cp), "cm_dg_lsrk_step_table")


def cm_dg_filter(ctx, Q_dev):
    _check(_load().cm_dg_filter(ctx, _dptr(Q_dev)), "cm_dg_filter")


def cm_dg_diagnostics(ctx, Q_dev):
    d = _Diag()
    _check(_load().cm_dg_diagnostics(ctx, _dptr(Q_dev), C.byref(d)), "cm_dg_diagnostics")
    return {k: getattr(d, k) for k, _ in _Diag._fields_}


STATIC_MAX_ELEM = 65536   # CM_DG_STATIC_MAX_ELEM


def cm_dg_diagnostics_static(cfg, n_elem, field_stride, Q_dev, J_dev, z_dev, stream=None):
    """Conservation sums of Q_dev without a ctx and without device allocation (include/cm_dg.h: for callers that cannot
    cudaMalloc, e.g. beside a memory pool that owns the GPU).  cfg supplies N, nvar and the Table-1 constants; J_dev and z_dev
    are per-node arrays in the library layout (cm_dg_metrics' J, row 2 of cm_dg_coords).  Marshalling only."""
    d = _StaticDesc(N=int(cfg["N"]), nvar=int(cfg.get("nvar", 5)), n_elem=int(n_elem), field_stride=int(field_stride))
    for k in ("R_d", "c_vd", "R_v", "c_vv", "T_0", "I_v0", "grav"):
        setattr(d, k, float(cfg[k]))
    out = _Diag()
    sp = C.c_void_p(int(stream.cuda_stream)) if stream is not None else C.c_void_p(0)
    _check(_load().cm_dg_diagnostics_static(C.byref(d), _dptr(Q_dev), _dptr(J_dev), _dptr(z_dev), sp, C.byref(out)),
           "cm_dg_diagnostics_static")
    return {k: getattr(out, k) for k, _ in _Diag._fields_}


NPROF = 20   # CM_DG_NPROF


def cm_dg_profiles(ctx, Q_dev, out_host):
    """out_host: numpy float64 [nlev][NPROF] (nlev >= Ez * Nq)."""
    assert out_host.ndim == 2 and out_host.shape[1] == NPROF
    _check(_load().cm_dg_profiles(ctx, _dptr(Q_dev), _hptr(out_host), int(out_host.shape[0])), "cm_dg_profiles")
    return out_host


def cm_dg_rhs_host(ctx, Q_host, dQ_host, t=0.0):
    _check(_load().cm_dg_rhs_host(ctx, _hptr(Q_host), _hptr(dQ_host), float(t)), "cm_dg_rhs_host")


def cm_dg_lsrk_step_host(ctx, Q_host, t, dt, nsteps):
    _check(_load().cm_dg_lsrk_step_host(ctx, _hptr(Q_host), float(t), float(dt), int(nsteps)), "cm_dg_lsrk_step_host")


def cm_dg_profile_begin(ctx):
    _check(_load().cm_dg_profile_begin(ctx), "cm_dg_profile_begin")


def cm_dg_profile_end(ctx):
    s = _KStats()
    _check(_load().cm_dg_profile_end(ctx, C.byref(s)), "cm_dg_profile_end")
    return {k: getattr(s, k) for k, _ in _KStats._fields_}


def cm_dg_destroy(ctx):
    _load().cm_dg_destroy(ctx)


class CmDg:
    """Owns one ctx; allocates state arrays with torch on the current CUDA device."""

    def __init__(self, cfg, stream=None, tuning=None):
        import torch
        self.torch = torch
        self.cfg = cfg
        self.ctx = cm_dg_setup(cfg, stream, tuning)
        self.n_elem, self.np, self.stride, self.lex_of_elem = cm_dg_layout(self.ctx)
        self.nvar = int(cfg.get("nvar", 5))
        self.device = torch.device("cuda", torch.cuda.current_device())

    def close(self):
        if getattr(self, "ctx", None):
            cm_dg_destroy(self.ctx); self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- layout helpers (host side, numpy): lexicographic AoS <-> library SoA
    def pack(self, Q_lex):
        """Q_lex[Ne, Np, nv] (lexicographic elements) -> numpy [nv, stride] in library layout."""
        nv = Q_lex.shape[-1]
        out = np.zeros((nv, self.stride))
        out[:, : self.n_elem * self.np] = np.moveaxis(Q_lex[self.lex_of_elem], -1, 0).reshape(nv, -1)
        return out

    def unpack(self, A):
        """numpy [nv, stride] in library layout -> [Ne, Np, nv] lexicographic."""
        nv = A.shape[0]
        lib = np.moveaxis(A[:, : self.n_elem * self.np].reshape(nv, self.n_elem, self.np), 0, -1)
        out = np.empty_like(lib)
        out[self.lex_of_elem] = lib
        return out

    def to_device(self, Q_lex):
        return self.torch.from_numpy(self.pack(Q_lex)).to(self.device)

    def to_host(self, T):
        return self.unpack(T.cpu().numpy())

    def empty(self, nfields):
        return self.torch.zeros((nfields, self.stride), dtype=self.torch.float64, device=self.device)

    # ---- the C entry points
    def coords(self):
        x = self.empty(3); cm_dg_coords(self.ctx, x); return x

    def metrics(self):
        Ja = self.empty(9); J = self.empty(1); cm_dg_metrics(self.ctx, Ja, J); return Ja, J

    def gradient(self, Q):
        G = self.empty(15); cm_dg_gradient(self.ctx, Q, G); return G

    def rhs(self, Q, dQ=None, t=0.0):
        if dQ is None:
            dQ = self.empty(self.nvar)
        cm_dg_rhs(self.ctx, Q, dQ, t)
        return dQ

    def lsrk_step(self, Q, dt, nsteps=1, t=0.0):
        cm_dg_lsrk_step(self.ctx, Q, t, dt, nsteps)
        return Q

    def lsrk_step_table(self, Q, dt, nsteps, A, B, t=0.0):
        cm_dg_lsrk_step_table(self.ctx, Q, t, dt, nsteps, A, B)
        return Q

    def filter(self, Q):
        cm_dg_filter(self.ctx, Q)
        return Q

    def diagnostics(self, Q):
        return cm_dg_diagnostics(self.ctx, Q)

    def profiles(self, Q):
        """Density-weighted horizontal statistics (App. B): numpy [Ez * Nq][NPROF]."""
        out = np.zeros((int(self.cfg["ne"][2]) * (int(self.cfg["N"]) + 1), NPROF))
        return cm_dg_profiles(self.ctx, Q, out)

    def rhs_host(self, Q_host, dQ_host, t=0.0):
        cm_dg_rhs_host(self.ctx, Q_host, dQ_host, t)

    def lsrk_step_host(self, Q_host, dt, nsteps=1, t=0.0):
        cm_dg_lsrk_step_host(self.ctx, Q_host, t, dt, nsteps)

    def profile_begin(self):
        cm_dg_profile_begin(self.ctx)

    def profile_end(self):
        return cm_dg_profile_end(self.ctx)
