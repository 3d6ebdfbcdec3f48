"""CPU-side checks of the boundary: libmcdc.so builds/loads without a GPU, exports every symbol that
include/mcdc.h declares, and fails loudly (no CPU fallback) when there is no device."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def M():
    from paper_2409_04668_b200 import build as b
    b.build()
    import paper_2409_04668_b200 as M
    return M


def _declared_symbols():
    txt = open(os.path.join(ROOT, "include", "mcdc.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(mcdc_[a-z_0-9]+)\s*\(", txt)))


def test_header_symbols_are_exported(M):
    decl = _declared_symbols()
    assert "mcdc_problem_create" in decl and "mcdc_run" in decl and "mcdc_tallies_get" in decl
    L = ctypes.CDLL(M.lib_path())
    for s in decl:
        assert hasattr(L, s), f"{s} declared in include/mcdc.h but not exported"
    assert sorted(M.EXPORTED_SYMBOLS) == decl


def test_binding_has_the_same_names(M):
    for s in _declared_symbols():
        if s in ("mcdc_last_cuda_error",):
            continue
        assert hasattr(M, s), s


def test_strerror_and_version(M):
    assert M.mcdc_strerror(0) == "ok"
    assert "overflow" in M.mcdc_strerror(-6)
    assert "sm_100a" in M.mcdc_version()


def test_library_does_not_link_torch_or_the_oracle(M):
    import subprocess
    out = subprocess.run(["ldd", M.lib_path()], capture_output=True, text=True).stdout
    assert "torch" not in out and "oracle" not in out
    # the product package never imports the oracle
    for fn in os.listdir(os.path.join(ROOT, "paper_2409_04668_b200")):
        if fn.endswith(".py"):
            src = open(os.path.join(ROOT, "paper_2409_04668_b200", fn)).read()
            assert "import oracle" not in src and "from oracle" not in src


def test_no_cpu_fallback_without_a_device(M):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from workloads import configs as W
    p = W.config0_infinite_medium(n_histories=100, n_batches=1)
    with pytest.raises(M.McdcError) as e:
        M.mcdc_problem_create(p)
    assert e.value.code == -7
    with pytest.raises(RuntimeError):
        M.Problem(p)


def test_description_is_validated_before_any_cuda_call(M):
    from workloads import configs as W
    p = W.config0_infinite_medium(n_histories=100, n_batches=1)
    p.sigma_c = p.sigma_c.copy(); p.sigma_c[0, 0] = 0.25            # Sigma_t != Sigma_c + Sigma_s + Sigma_f
    with pytest.raises(M.McdcError) as e:
        M.mcdc_problem_create(p)
    assert e.value.code == -2
    p = W.config0_infinite_medium(n_histories=100, n_batches=1)
    p.hs_surface = p.hs_surface.copy(); p.hs_surface[0] = 17         # surface id out of range
    with pytest.raises(M.McdcError) as e:
        M.mcdc_problem_create(p)
    assert e.value.code == -3
    p = W.config0_infinite_medium(n_histories=100, n_batches=1)
    p.time_edges = p.time_edges.copy(); p.time_edges[3] = p.time_edges[2]   # not strictly increasing
    with pytest.raises(M.McdcError) as e:
        M.mcdc_problem_create(p)
    assert e.value.code == -9
    p = W.config0_infinite_medium(n_histories=100, n_batches=1)
    p.census_times = p.census_times[:-1].copy() * 0 + np.arange(1, 20) * -1.0   # census before the source time
    with pytest.raises(M.McdcError) as e:
        M.mcdc_problem_create(p)
    assert e.value.code == -9
