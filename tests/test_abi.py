"""The C-ABI library loads on a CPU-only box and exports every symbol include/dhp.h declares
(no compute calls here: those need a GPU and live in test_gpu_parity.py)."""
import os
import re

from paper_2207_14276_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "dhp.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dhp_[a-z_0-9]+)\s*\(", text)))


def test_header_and_binding_agree():
    assert declared_symbols() == sorted(binding.SYMBOLS)


def test_library_builds_loads_and_exports_everything():
    from paper_2207_14276_b200 import build
    build.build()
    lib = binding.load_library()
    for name in declared_symbols():
        assert hasattr(lib, name), name
    assert b"sm_100a" in lib.dhp_version()
    assert lib.dhp_strerror(-3).decode().startswith("periodic box")
    assert lib.dhp_strerror(0) == b"ok"


def test_params_struct_matches_header():
    import ctypes
    # 6 scalars, shf_r[16], shf_a[8], shf_z[8], n_shf_a, n_shf_z (include/dhp.h: dhp_params)
    assert ctypes.sizeof(binding.DhpParams) == 4 * (6 + 16 + 8 + 8 + 2)
    from paper_2207_14276_b200 import workloads as W
    for p, grid in ((W.default_params(), (8, 4)), (W.ani1x_params(), (4, 8))):
        q = binding.make_params(p)
        assert (q.n_shf_a, q.n_shf_z) == grid and abs(q.shf_z[grid[1] - 1] - float(p.shf_z[-1])) < 1e-7


def test_no_cpu_fallback_without_gpu():
    import pytest
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(binding.DhpError):
        binding.Dhp(16)


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2207_14276_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "liboracle" not in src, f


def test_experiment_builds_cannot_pass_for_the_default_library(monkeypatch):
    """DHP_NVCC_EXTRA injects timing-experiment macros, some of which give wrong results by design.  The flags are
    compiled into dhp_version() and kept in a stamp beside the library: a library built with other flags than the current ones
    is stale (rebuilt by build()), and the default build says nothing about extra flags (binding.load_library refuses one
    that does unless DHP_ALLOW_EXPERIMENT=1)."""
    from paper_2207_14276_b200 import build
    build.build()
    assert not build._stale()
    assert b"extra flags" not in binding.load_library().dhp_version()
    assert open(build.STAMP).read() == ""
    monkeypatch.setattr(build, "EXTRA", ["-DMID_TRACE=1"])
    assert build._stale()
