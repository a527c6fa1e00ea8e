"""Bitwise repeatability of every kernel variant (the race detector of last resort where compute-sanitizer is closed,
profiles/r2_sanitizer.md): each case runs one cm_dg_rhs and two cm_dg_lsrk_step calls THREE times from the same input, and
the horizontal statistics twice; the results must agree bit for bit.  The kernels have no atomics and a fixed summation
order, so any difference is an ordering bug in the mbarrier / cp.async / named-barrier protocol.  Covers the row-sweep,
CTA-per-element and stored-metric kernels, both L2-prefetch settings, walls and periodic sides, dry and moist, every closure,
the sponge, the element filter, HLLC / Roe, surface fluxes and the saturation adjustment.

Under the sanitizer (when a pool allows it):
    compute-sanitizer --tool memcheck  python -m pytest tests/test_gpu_repeatability.py -m gpu -x -q
    compute-sanitizer --tool racecheck python -m pytest tests/test_gpu_repeatability.py -m gpu -x -q"""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2110_00853_b200 as pkg
    return pkg


def _c1(**kw):
    return W.config1(ne=(4, 4, 4), N=4), kw


def _c3(**kw):
    return W.config3(ne=(5, 4, 6), N=4, hi=(1000.0, 800.0, 1125.0)), kw


def _c4(**kw):
    return W.config4(ne=(14, 1, 6), N=4), kw


def _c5(N=4, **kw):
    return W.config5(ne=(6, 5, 7), N=N, hi=(375.0, 312.5, 3000.0)), kw


_FLUX = dict(drag_cd=1.3e-3, lhf_bottom=147.2, evap_bottom=5.9e-5)
CASES = [
    ("config1 row-sweep", _c1, {}, None), ("config1 cm7", _c1, {}, {"kernel": 7}), ("config1 stored-metric", _c1, {}, {"kernel": 2}),
    ("config3 row-sweep", _c3, {}, None), ("config3 rows of 1", _c3, {}, {"row_len": 1}),
    ("config5 row-sweep", _c5, {}, None), ("config5 cm7 ahead 2/3", _c5, {}, {"kernel": 7, "ahead_t": 2, "ahead_g": 3}),
    ("config5 cm7 no prefetch", _c5, {}, {"kernel": 7, "ahead_t": 0, "ahead_g": 0}),
    ("config5 stored-metric", _c5, {}, {"kernel": 2}), ("config5 N=3", _c5, {"N": 3}, None), ("config5 N=5", _c5, {"N": 5}, None),
    ("config5 N=6 (cm7)", _c5, {"N": 6}, None),
    ("config4 terrain", _c4, {}, None), ("config4 terrain + closure", _c4, {"sgs": 1}, None),
    ("config5 Vreman + Richardson", _c5, {"sgs": 2, "richardson": 1}, None),
    ("config4 sponge + filter", _c4, dict(sponge_alpha=0.4, sponge_zs=2500.0, u_relax=(10.0, 0.0, 0.0), filter_order=64), None),
    ("config5 filter", _c5, {"filter_order": 64}, None), ("config3 HLLC", _c3, {"riemann": 1}, None), ("config3 Roe", _c3, {"riemann": 2}, None),
    ("config5 surface fluxes", _c5, _FLUX, None), ("config5 surface fluxes cm7", _c5, _FLUX, {"kernel": 7}),
    ("config5 saturation adjustment", _c5, {"satadj": 1}, None),
    ("config5 long rows", lambda **kw: (W.config5(ne=(32, 4, 3), N=4, hi=(2000.0, 250.0, 187.5)), kw), {}, None),
]


@pytest.mark.parametrize("name,make,over,tuning", CASES, ids=[c[0].replace(" ", "_") for c in CASES])
def test_bitwise_repeatable(P, name, make, over, tuning):
    import torch
    (cfg, Q, dt), kw = make(**over)
    cfg = dict(cfg, **kw)
    g = P.CmDg(cfg, tuning=tuning)
    runs = []
    for _ in range(3):
        Qd = g.to_device(Q)
        dQ = g.rhs(Qd).clone()
        g.lsrk_step(Qd, dt, 2)
        runs.append((dQ, Qd))
    d = g.diagnostics(runs[0][1])
    prof = [g.profiles(runs[0][1]) for _ in range(2)]
    assert bool(torch.isfinite(runs[0][0]).all()) and d["n_nonfinite"] == 0, name
    assert np.array_equal(prof[0], prof[1]), name
    for r in runs[1:]:
        assert bool((r[0] == runs[0][0]).all()) and bool((r[1] == runs[0][1]).all()), name
    g.close()
