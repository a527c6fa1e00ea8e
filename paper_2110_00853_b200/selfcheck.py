"""Small end-to-end run of every kernel variant, meant to be run under compute-sanitizer (profiles/r2_sanitizer.md):

    compute-sanitizer --tool memcheck  python -m paper_2110_00853_b200.selfcheck
    compute-sanitizer --tool racecheck python -m paper_2110_00853_b200.selfcheck

Where the sanitizer is not available the same run is its own race detector of last resort: every case is executed
THREE times from the same input and the results must agree bit for bit (the kernels have no atomics and a fixed
summation order, so any difference is an ordering bug in the mbarrier / cp.async / barrier protocol).

One cm_dg_rhs and two cm_dg_lsrk_step calls per case on small seeded meshes: the row-sweep, CTA-per-element and
stored-metric kernels, both L2-prefetch settings, walls and periodic sides, dry and moist, every closure, the sponge,
the element filter, HLLC / Roe, surface fluxes, the saturation adjustment and the horizontal statistics.  Prints one line per case; exits non-zero on a non-finite result.
"""
import sys

import numpy as np


def main():
    import torch
    import workloads as W
    from . import CmDg
    assert torch.cuda.is_available(), "selfcheck needs a CUDA device"
    c1 = lambda **kw: (W.config1(ne=(4, 4, 4), N=4), kw)
    c3 = lambda **kw: (W.config3(ne=(5, 4, 6), N=4, hi=(1000.0, 800.0, 1125.0)), kw)
    c4 = lambda **kw: (W.config4(ne=(14, 1, 6), N=4), kw)
    c5 = lambda N=4, **kw: (W.config5(ne=(6, 5, 7), N=N, hi=(375.0, 312.5, 3000.0)), kw)
    cases = [
        ("config1 row-sweep", c1(), None), ("config1 cm7", c1(), {"kernel": 7}), ("config1 stored-metric", c1(), {"kernel": 2}),
        ("config3 row-sweep", c3(), None), ("config3 rows of 1", c3(), {"row_len": 1}),
        ("config5 row-sweep", c5(), None), ("config5 cm7 ahead 2/3", c5(), {"kernel": 7, "ahead_t": 2, "ahead_g": 3}),
        ("config5 cm7 no prefetch", c5(), {"kernel": 7, "ahead_t": 0, "ahead_g": 0}),
        ("config5 stored-metric", c5(), {"kernel": 2}), ("config5 N=3", c5(N=3), None), ("config5 N=5", c5(N=5), None),
        ("config5 N=6 (cm7)", c5(N=6), None),
        ("config4 terrain", c4(), None), ("config4 terrain + closure", c4(sgs=1), None),
        ("config5 Vreman + Richardson", c5(sgs=2, richardson=1), None),
        ("config4 sponge + filter", c4(sponge_alpha=0.4, sponge_zs=2500.0, u_relax=(10.0, 0.0, 0.0), filter_order=64), None),
        ("config5 filter", c5(filter_order=64), None), ("config3 HLLC", c3(riemann=1), None), ("config3 Roe", c3(riemann=2), None),
        ("config5 surface fluxes", c5(drag_cd=1.3e-3, lhf_bottom=147.2, evap_bottom=5.9e-5), None),
        ("config5 surface fluxes cm7", c5(drag_cd=1.3e-3, lhf_bottom=147.2, evap_bottom=5.9e-5), {"kernel": 7}),
        ("config5 saturation adjustment", c5(satadj=1), None),
        ("config5 long rows", (W.config5(ne=(32, 4, 3), N=4, hi=(2000.0, 250.0, 187.5)), {}), None),
    ]
    bad = 0
    for name, ((cfg, Q, dt), over), tuning in cases:
        cfg = dict(cfg, **over)
        g = CmDg(cfg, tuning=tuning)
        runs = []
        for _ in range(3):
            Qd = g.to_device(Q)
            dQ = g.rhs(Qd).clone()
            g.lsrk_step(Qd, dt, 2)
            runs.append((dQ, Qd))
        d = g.diagnostics(runs[0][1])
        prof = [g.profiles(runs[0][1]) for _ in range(2)]
        same_prof = bool(np.array_equal(prof[0], prof[1]))
        finite = bool(torch.isfinite(runs[0][0]).all()) and d["n_nonfinite"] == 0
        same = same_prof and all(bool((r[0] == runs[0][0]).all()) and bool((r[1] == runs[0][1]).all()) for r in runs[1:])
        bad += 0 if (finite and same) else 1
        print("%-32s %s %s  mass %.12e" % (name, "finite" if finite else "NON-FINITE", "bitwise-repeatable" if same else "NOT REPEATABLE", d["mass"]))
        g.close()
    return 1 if bad else 0


if __name__ == "__main__":
    sys.exit(main())
