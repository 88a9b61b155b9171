"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every symbol
include/tddp4.h declares; the product path has no CPU fallback; the workload tables are consistent."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_1702_06735_b200 import binding, build, workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    return build.build_library()


def test_library_exports_every_declared_symbol(lib_path):
    header = open(os.path.join(ROOT, "include", "tddp4.h")).read()
    declared = set(re.findall(r"\b(tddp4_[a-z_0-9]+)\s*\(", header))
    declared -= {"tddp4_status"}
    assert declared == set(binding.SYMBOLS), declared ^ set(binding.SYMBOLS)
    lib = ctypes.CDLL(lib_path)
    for name in declared:
        assert hasattr(lib, name), name
    lib.tddp4_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.tddp4_version()


def test_library_has_sm100a_code(lib_path):
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", lib_path], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        binding.Tddp4(W.config(1).model)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1702_06735_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "tddp4_oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import binding" not in src and "paper_1702_06735_b200.binding" not in src, f
            assert "libtddp4.so" not in src and "#include \"../paper" not in src, f


def test_config_tables():
    c1, c2, c3, c5 = W.config(1), W.config(2), W.config(3), W.config(5)
    assert (c1.model.n_terms, c1.model.n_couplings, c1.n_data, c1.n_norm) == (3, 3, 1000, 10000)
    assert (c2.model.n_terms, c2.model.n_couplings, c2.n_data, c2.n_norm) == (8, 8, 50000, 500000)
    assert (c3.model.n_terms, c3.model.n_couplings, c3.n_data, c3.n_norm) == (16, 8, 1000000, 4000000)
    assert c5.model.use_resolution == 1 and c5.model.t_hi == 4.0
    # ordering B is ordering A with the identical pions exchanged, same coupling
    m = c3.model
    for k in range(0, 16, 2):
        assert m.term_coupling[k] == m.term_coupling[k + 1]
        a, b = m.term_perm[k], m.term_perm[k + 1]
        assert tuple({1: 3, 3: 1}.get(v, v) for v in a) == b


def test_trajectories_are_seeded_and_shaped():
    mdl = W.config(3).model
    p0 = W.initial_params(mdl)
    tr = W.trajectory(mdl, p0, 50, "minuit")
    tr2 = W.trajectory(mdl, p0, 50, "minuit")
    assert all(np.array_equal(a.c, b.c) and np.array_equal(a.mass, b.mass) for a, b in zip(tr, tr2))
    co = W.trajectory(mdl, p0, 20, "coupling_only")
    assert all(np.array_equal(p.mass, p0.mass) and np.array_equal(p.width, p0.width) for p in co)
    al = W.trajectory(mdl, p0, 5, "all")
    assert all(not np.array_equal(p.mass, p0.mass) for p in al)
    assert np.all(np.abs(p0.c) >= 0.5) and np.all(np.abs(p0.c) <= 2.0)
