"""cm_dg_diagnostics_static: the conservation sums for callers that cannot allocate device memory.

Some users of this library hold a state array on the GPU but cannot call cudaMalloc, so they cannot create a ctx with
cm_dg_setup: the application's memory pool (a framework's caching allocator, an arena) already owns the whole device, or
they are a monitor attached to somebody else's run without a memory budget, or they sit in a loop where cudaMalloc's
device-wide synchronisation is not acceptable.  For them the library carries one built-in scratch array
(CM_DG_STATIC_SCRATCH_BYTES, at most CM_DG_STATIC_MAX_ELEM elements) and this one entry point that uses it.

Checked here: the built-in-scratch entry point gives the same sums as cm_dg_diagnostics (the ctx path, scratch from
cudaMalloc) within the 1e-12 of test_diagnostics_parity, on calls made back to back that share the array (a large mesh, then
a smaller one with another state and geometry, then the first again); free device memory does not move across the calls;
a mesh beyond the limit is refused with a message that names the limit.

This file sorts last on purpose (pytest -x would otherwise let a failure here hide the tests behind it), and it has to pass
both alone in a fresh process and after the rest of the suite."""
import numpy as np
import pytest

from parity_util import small_config

pytestmark = pytest.mark.gpu

KEYS = ("mass", "energy", "water", "kinetic", "max_wavespeed", "volume")
TOL = 1e-12   # the bar of test_diagnostics_parity


@pytest.fixture(scope="module")
def P():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2110_00853_b200 as pkg
    return pkg


class _Case:
    """A ctx (the existing path) plus the three caller-owned arrays the ctx-free entry point reads."""

    def __init__(self, P, k, nsteps):
        self.cfg, Q, dt = small_config(k)
        self.g = P.CmDg(self.cfg)
        self.Q = self.g.to_device(Q)
        if nsteps:
            self.g.lsrk_step(self.Q, dt, nsteps)           # a state with flow in it
        self.J = self.g.metrics()[1][0].contiguous()
        self.z = self.g.coords()[2].contiguous()

    def ctx_path(self, P):
        return self.g.diagnostics(self.Q)

    def static_path(self, P, Q=None):
        return P.cm_dg_diagnostics_static(self.cfg, self.g.n_elem, self.g.stride, self.Q if Q is None else Q, self.J, self.z)


def _agree(d, ref, label):
    for key in KEYS:
        assert abs(d[key] - ref[key]) <= TOL * max(abs(ref[key]), 1e-300), (label, key, d[key], ref[key])
    assert d["n_nonfinite"] == ref["n_nonfinite"], label
    assert d["min_node_dx"] == 0.0                         # documented: the ctx-free call does not know the mesh


def test_static_scratch_matches_ctx_path_on_consecutive_calls(P):
    import torch
    big = _Case(P, 5, 3)       # moist, flat brick, Smagorinsky
    small = _Case(P, 4, 2)     # dry, terrain-following (stored metrics), fewer elements
    assert small.g.n_elem < big.g.n_elem, "the second call must leave stale sums of the first one behind it"
    ref_big, ref_small = big.ctx_path(P), small.ctx_path(P)
    assert ref_big["mass"] != ref_small["mass"]

    first = big.static_path(P)                             # first call on this device: looks up the built-in array
    _agree(first, ref_big, "call 1 (large mesh)")
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    second = small.static_path(P)                          # straight after it, on the same array
    third = big.static_path(P)
    fourth = big.static_path(P)
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]
    _agree(second, ref_small, "call 2 (small mesh after large)")
    _agree(third, ref_big, "call 3 (large mesh again)")
    assert third == first and fourth == first, "same input, same array: the sums are formed in a fixed order"
    assert free_after == free_before, "the entry point must not take device memory (%d -> %d)" % (free_before, free_after)

    # a non-finite value is counted, and the count does not stick to the array for the next call
    Qbad = big.Q.clone(); Qbad[4, 17] = float("inf")
    assert big.static_path(P, Qbad)["n_nonfinite"] == 1 == big.g.diagnostics(Qbad)["n_nonfinite"]
    _agree(big.static_path(P), ref_big, "call after a non-finite state")


def test_static_scratch_on_a_side_stream(P):
    import torch
    c = _Case(P, 2, 1)
    ref = c.ctx_path(P)
    torch.cuda.synchronize()
    s = torch.cuda.Stream()
    d = P.cm_dg_diagnostics_static(c.cfg, c.g.n_elem, c.g.stride, c.Q, c.J, c.z, stream=s)
    _agree(d, ref, "side stream")


def test_static_scratch_refuses_meshes_beyond_the_limit(P):
    c = _Case(P, 1, 0)
    with pytest.raises(P.CmDgError, match="CM_DG_STATIC_MAX_ELEM = 65536"):
        P.cm_dg_diagnostics_static(c.cfg, P.binding.STATIC_MAX_ELEM + 1, 2 ** 40, c.Q, c.J, c.z)
    with pytest.raises(P.CmDgError, match="field_stride"):
        P.cm_dg_diagnostics_static(c.cfg, c.g.n_elem, c.g.n_elem * c.g.np - 1, c.Q, c.J, c.z)
    _agree(c.static_path(P), c.ctx_path(P), "after refused calls")
