"""cm_dg_lsrk_step replays a time step from a CUDA graph once the same (Q_dev, dt, table) has been seen twice: the replayed
steps must be bit-identical to kernel-by-kernel launches (same kernels, same arguments), survive a change of the state
array or dt (re-capture), coexist with the per-launch profiling events, and not be slower on a launch-bound mesh."""
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
    assert times["graph"] <= 1.5 * times["plain"]
