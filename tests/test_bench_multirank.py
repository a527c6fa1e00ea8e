"""The N > 1 path of bench.py on CPU: two gloo ranks, each with its own replica timing; the whole-job value must use
the MAX time over ranks and count every rank's nodes (weak scaling, "replicas only": no data-path collective)."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms_local = 10.0 + 5.0 * rank                      # rank 1 is the slower replica
    value, ms = bench.whole_job_value(1000, 4, ms_local, world, dist, torch.device("cpu"))
    mx = bench.max_over_ranks(rank, dist, torch.device("cpu"))
    dist.barrier()
    out.put((rank, value, ms, mx))
    dist.destroy_process_group()


def test_whole_job_value_is_max_over_ranks():
    world, port = 2, 29517 + os.getpid() % 1000
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, value, ms, mx in res:
        assert ms == 15.0                              # max over ranks
        assert mx == 1.0
        assert abs(value - world * 1000 * 5 * 4 / 15.0e-3) < 1e-6 * value


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    value, ms = bench.whole_job_value(1000, 2, 8.0, 1, None, None)
    assert ms == 8.0 and abs(value - 1000 * 5 * 2 / 8.0e-3) < 1e-9 * value


def test_bench_legs_are_well_formed():
    """Host logic of bench.py's further workloads: every NEXT-row leg exists, builds its config on the shared 48x48x48 cut of
    config 5 with exactly the option it names switched on, and carries a positive algorithmic byte count."""
    import bench
    import workloads as W
    assert set(bench.NEXT_LEGS) <= set(bench.LEGS)
    want = {"c5_vreman": {"sgs": 2, "richardson": 1}, "c5_hllc": {"riemann": 1}, "c5_roe": {"riemann": 2},
            "c5_satadj": {"satadj": 1}, "c5_sponge_filter": {"filter_order": 64}, "c5_surface": {"drag_cd": 1.3e-3}}
    base = None
    for name in bench.NEXT_LEGS:
        make, steps, label, sb = bench.LEGS[name]
        cfg, Q, dt = make(W)
        assert tuple(cfg["ne"]) == (48, 48, 48) and cfg["N"] == 4 and cfg["nvar"] == 6 and steps >= 3
        for k, v in want[name].items():
            assert cfg[k] == v, (name, k)
        assert bench.stage_bytes(*sb) > 0 and "48x48x48" in label
        base = Q if base is None else base
        assert Q is base                                  # one seeded state shared by the legs
