"""CPU checks of the boundary: the C-ABI library builds for sm_100a, loads, exports every symbol that
include/cm_dg.h declares, and fails loudly (no CPU fallback) when there is no CUDA device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2110_00853_b200 import build
    path = build.build()
    return ctypes.CDLL(path)


def test_header_symbols_are_exported(lib):
    text = open(os.path.join(ROOT, "include", "cm_dg.h")).read()
    names = set(re.findall(r"\b(cm_dg_[a-z_]+)\s*\(", text))
    assert {"cm_dg_setup", "cm_dg_rhs", "cm_dg_lsrk_step", "cm_dg_diagnostics"} <= names
    for n in names:
        assert hasattr(lib, n), n
    from paper_2110_00853_b200 import binding
    assert set(binding.EXPORTS) == names


def test_library_is_compiled_for_sm100a():
    import subprocess
    from paper_2110_00853_b200 import binding
    out = subprocess.run(["cuobjdump", "--list-elf", binding.library_path()], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("only meaningful on a machine without a GPU")
    import paper_2110_00853_b200 as P
    import workloads as W
    cfg, Q, dt = W.config1()
    with pytest.raises(P.CmDgError, match="no CUDA device"):
        P.cm_dg_setup(cfg)


def test_argument_validation_precedes_device_use():
    import paper_2110_00853_b200 as P
    import workloads as W
    cfg, Q, dt = W.config1()
    bad = dict(cfg); bad["N"] = 1
    with pytest.raises(P.CmDgError, match="polynomial order"):
        P.cm_dg_setup(bad)
    bad = dict(cfg); bad["bc"] = (0, 2, 0)
    with pytest.raises(P.CmDgError, match="bc"):
        P.cm_dg_setup(bad)
    # prescribed evaporation enters rho and rho*q_tot: a dry state (nvar == 5) cannot carry it
    bad = dict(cfg); bad["bc"] = (0, 0, 1); bad["nvar"] = 5; bad["evap_bottom"] = 1e-5
    with pytest.raises(P.CmDgError, match="evap_bottom needs the moisture tracer"):
        P.cm_dg_setup(bad)


def test_refused_setup_clears_the_handle():
    """*out is NULL after every refusal, also one caused by the tuning struct (checked first)."""
    import ctypes as C
    from paper_2110_00853_b200 import binding as B
    L = B._load()
    p = B._Params(); p.N = 4
    tn = B._Tuning(kernel=5, ahead_t=-1, ahead_g=-1)
    ctx = C.c_void_p(0xdead)
    assert L.cm_dg_setup_tuned(C.byref(p), C.byref(tn), None, C.byref(ctx)) == -1
    assert not ctx.value


def test_static_diagnostics_checks_its_limit_before_device_use():
    """cm_dg_diagnostics_static (built-in scratch array, for callers that cannot cudaMalloc) refuses a mesh beyond
    CM_DG_STATIC_MAX_ELEM with a message naming the limit, before anything touches a device."""
    import paper_2110_00853_b200 as P
    import workloads as W
    cfg, Q, dt = W.config1()
    text = open(os.path.join(ROOT, "include", "cm_dg.h")).read()
    assert int(re.search(r"#define CM_DG_STATIC_MAX_ELEM (\d+)", text).group(1)) == P.binding.STATIC_MAX_ELEM
    with pytest.raises(P.CmDgError, match="exceeds CM_DG_STATIC_MAX_ELEM = %d" % P.binding.STATIC_MAX_ELEM):
        P.cm_dg_diagnostics_static(cfg, P.binding.STATIC_MAX_ELEM + 1, 2 ** 40, 256, 256, 256)
    with pytest.raises(P.CmDgError, match="NULL"):
        P.cm_dg_diagnostics_static(cfg, 8, 8 * 125, 0, 256, 256)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2110_00853_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                s = open(os.path.join(dp, f)).read()
                assert "oracle" not in s.lower().replace("no cpu fallback", ""), os.path.join(dp, f)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            s = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2110_00853_b200" not in s and "cm_dg.h" not in s
