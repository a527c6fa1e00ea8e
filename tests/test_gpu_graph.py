"""cm_dg_lsrk_step replays a time step from a CUDA graph once the same (Q_dev, dt, table) has been seen twice: the replayed
steps must be bit-identical to kernel-by-kernel launches (same kernels, same arguments), survive a change of the state
array or dt (re-capture), coexist with the per-launch profiling events; the speed on a launch-bound mesh is printed, not gated (bench.py reports it)."""
import time

import numpy as np
import pytest

import workloads as W
from parity_util import small_config

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2110_00853_b200 as pkg
    return pkg


@pytest.mark.parametrize("k,over", [(2, {}), (5, {}), (4, {"filter_order": 64}), (5, {"sgs": 2, "richardson": 1})])
def test_graph_replay_is_bitwise_identical(P, k, over):
    import torch
    cfg, Q, dt = small_config(k)
    cfg = dict(cfg, **over)
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        ga = P.CmDg(cfg, stream=stream); gb = P.CmDg(cfg, stream=stream, tuning={"no_graph": 1})
        Qa, Qb = ga.to_device(Q), gb.to_device(Q)
        for _ in range(5):                                # call 1 launches directly, call 2 captures, calls 3-5 replay
            ga.lsrk_step(Qa, dt, 3); gb.lsrk_step(Qb, dt, 3)
        stream.synchronize()
        assert torch.equal(Qa, Qb)
        # another state array, another dt: new keys, captured again on their second use
        Qc, Qd = ga.to_device(Q), gb.to_device(Q)
        for _ in range(3):
            ga.lsrk_step(Qc, 0.5 * dt, 2); gb.lsrk_step(Qd, 0.5 * dt, 2)
        ga.lsrk_step(Qa, dt, 1); gb.lsrk_step(Qb, dt, 1)    # back to the first array: the cached graph no longer matches
        ga.lsrk_step(Qa, dt, 1); gb.lsrk_step(Qb, dt, 1)
        # profiling events switch the graph off for the calls in between
        ga.profile_begin(); ga.lsrk_step(Qa, dt, 2); ks = ga.profile_end(); gb.lsrk_step(Qb, dt, 2)
        assert ks["launches_tendency"] == 10
        ga.lsrk_step(Qa, dt, 2); gb.lsrk_step(Qb, dt, 2)
        stream.synchronize()
        assert torch.equal(Qc, Qd) and torch.equal(Qa, Qb)
    ga.close(); gb.close()


def test_graph_key_compares_the_whole_table(P):
    """Two 5-stage tables whose weighted sums sum_s (s+1)(A_s + 3 B_s) are equal (B_0 + d, B_1 - d/2) but whose
    coefficients differ: the second table must not replay the graph captured for the first one."""
    import torch
    cfg, Q, dt = small_config(2)
    A1 = np.array([0.0, -0.4, -1.2, -1.7, -1.5]); B1 = np.array([0.15, 0.38, 0.82, 0.70, 0.15])
    A2 = A1.copy(); B2 = B1.copy(); B2[0] += 0.01; B2[1] -= 0.005
    w = np.arange(1, 6)
    assert abs(np.sum(w * (A1 + 3 * B1)) - np.sum(w * (A2 + 3 * B2))) < 1e-15 and B1.sum() != B2.sum()
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        ga = P.CmDg(cfg, stream=stream); gb = P.CmDg(cfg, stream=stream, tuning={"no_graph": 1})
        Qa, Qb = ga.to_device(Q), gb.to_device(Q)
        for A, B in ((A1, B1), (A2, B2), (A1, B1)):
            for _ in range(3):                            # direct, capture, replay
                ga.lsrk_step_table(Qa, dt, 1, A, B); gb.lsrk_step_table(Qb, dt, 1, A, B)
            stream.synchronize()
            assert torch.equal(Qa, Qb)
    ga.close(); gb.close()


def test_graph_on_the_default_stream_falls_back(P):
    import torch
    cfg, Q, dt = small_config(2)
    ga = P.CmDg(cfg); gb = P.CmDg(cfg, tuning={"no_graph": 1})      # legacy default stream: cannot be captured
    Qa, Qb = ga.to_device(Q), gb.to_device(Q)
    for _ in range(4):
        ga.lsrk_step(Qa, dt, 2); gb.lsrk_step(Qb, dt, 2)
    torch.cuda.synchronize()
    assert torch.equal(Qa, Qb)
    ga.close(); gb.close()


def test_graph_is_not_slower_on_a_launch_bound_mesh(P):
    import torch
    cfg, Q, dt = W.config2()                             # 40x1x20 elements, 100 k nodes: ~10 us kernels
    stream = torch.cuda.Stream()
    times = {}
    with torch.cuda.stream(stream):
        for name, tun in (("graph", None), ("plain", {"no_graph": 1})):
            g = P.CmDg(cfg, stream=stream, tuning=tun)
            Qd = g.to_device(Q)
            for _ in range(3):
                g.lsrk_step(Qd, dt, 20)
            stream.synchronize()
            best = 1e9
            for _ in range(3):                           # best of three: the bound below must not depend on a noisy box
                t0 = time.perf_counter()
                for _ in range(10):
                    g.lsrk_step(Qd, dt, 20)
                stream.synchronize()
                best = min(best, (time.perf_counter() - t0) / 200)
            times[name] = best
            g.close()
    print("config 2, seconds per LSRK54 step: %r" % times)
    # Not a gate: a wall-clock ratio on a shared box is not a property of the code.  The measured graph / plain-launch step
    # times are reported by bench.py (roofline.c2_ms_per_step_graph / _no_graph and the c3, c4 pair); here a slower graph
    # only leaves a warning in the test log.
    if times["graph"] > 1.5 * times["plain"]:
        import warnings
        warnings.warn("CUDA-graph replay was slower than plain launches on config 2: %r" % times)
