"""CPU-side build check of the run-time specialised kernels (gram_jit.cuh, colnll_jit.cuh, gen_jit.cuh): the text tddp4_create hands
to NVRTC -- the generated prelude of model tables + the kernel file -- is obtained through the C-ABI
(tddp4_jit_source, no device needed) for every workload model and compiled here for sm_100a with NVRTC.  The cubins must
keep the lineshapes in registers (no local memory), and the Gram pass must contain fp64 tensor-core instructions."""
import os
import re
import subprocess

import pytest

from paper_1702_06735_b200 import binding, build, workloads as W

nvrtc = pytest.importorskip("cuda.bindings.nvrtc")


@pytest.fixture(scope="module", autouse=True)
def _lib():
    build.build_library()


def compile_sm100a(source, name, tmp_path):
    names = {b"jit_shared.cuh": 2, b"nll_shared.cuh": 3, b"tables.h": 5, b"device_math.cuh": 6}
    headers = [binding.jit_source(W.config(1).model, what).encode() for what in names.values()]
    err, prog = nvrtc.nvrtcCreateProgram(source.encode(), name.encode(), len(names), headers, list(names))
    assert err == nvrtc.nvrtcResult.NVRTC_SUCCESS
    opts = [b"--gpu-architecture=sm_100a", b"--std=c++17", b"-lineinfo"]
    (res,) = nvrtc.nvrtcCompileProgram(prog, len(opts), opts)
    _, n = nvrtc.nvrtcGetProgramLogSize(prog)
    log = b" " * n
    nvrtc.nvrtcGetProgramLog(prog, log)
    assert res == nvrtc.nvrtcResult.NVRTC_SUCCESS, log.decode()
    _, n = nvrtc.nvrtcGetCUBINSize(prog)
    cubin = b" " * n
    nvrtc.nvrtcGetCUBIN(prog, cubin)
    path = os.path.join(tmp_path, name + ".cubin")
    with open(path, "wb") as f:
        f.write(cubin)
    usage = subprocess.run(["cuobjdump", "-res-usage", path], capture_output=True, text=True).stdout
    sass = subprocess.run(["cuobjdump", "-sass", path], capture_output=True, text=True).stdout
    return usage, sass


def models():
    out = {f"C{i}": W.config(i).model for i in (1, 2, 3, 5)}
    out["flat"] = W.flat_model()
    return out


@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C5", "flat"])
def test_gram_pass_compiles_for_sm100a(name, tmp_path):
    mdl = models()[name]
    for weighted, gmode in ((False, 0), (True, 0), (False, 1), (False, 2)):
        usage, sass = compile_sm100a(binding.jit_source(mdl, 0, weighted, gmode), f"gram_{name}_{int(weighted)}{gmode}", str(tmp_path))
        assert "sm_100a" in sass
        m = re.search(r"REG:(\d+) STACK:(\d+)", usage)
        assert m and int(m.group(1)) <= 128, usage                               # two blocks per SM
        if gmode != 2:                                                           # (the incremental pass also holds the kept columns)
            assert int(m.group(2)) == 0 and "LDL" not in sass and "STL" not in sass, usage
        else:
            assert int(m.group(2)) <= 128, usage
        assert "DMMA" in sass                                                    # fp64 tensor cores
        # bulk L2 prefetch of the next tile (a constant-amplitude model streams no row at all: nothing to prefetch)
        if name != "flat":
            assert ("UBLKPF" in sass) == (gmode != 2)


@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C5", "flat"])
def test_data_pass_compiles_for_sm100a(name, tmp_path):
    mdl = models()[name]
    for mode in (0, 1, 2):
        usage, sass = compile_sm100a(binding.jit_source(mdl, 1, False, mode), f"colnll_{name}_{mode}", str(tmp_path))
        m = re.search(r"REG:(\d+) STACK:(\d+)", usage)
        assert m and int(m.group(1)) <= 128, usage
        if mode != 0:          # mode 0 calls sincos, whose large-argument path keeps a table on the stack
            assert int(m.group(2)) == 0 and "LDL" not in sass and "STL" not in sass, usage


@pytest.mark.parametrize("name", ["C1", "C3", "flat"])
def test_generator_kernel_compiles_for_sm100a(name, tmp_path):
    usage, sass = compile_sm100a(binding.jit_source(models()[name], 4), f"gen_{name}", str(tmp_path))
    m = re.search(r"REG:(\d+) STACK:(\d+)", usage)
    assert m and int(m.group(1)) <= 80, usage          # six blocks of 128 threads per SM
    assert "MUFU.RSQ64H" in sass and "MUFU.RCP64H" in sass


def test_prelude_states_the_model_tables():
    mdl = W.config(3).model
    src = binding.jit_source(mdl, 0)
    assert f"#define J_KC {mdl.n_couplings}\n" in src and f"#define J_NTERMS {mdl.n_terms}\n" in src
    last = [int(v) for v in re.search(r"J_LAST\[\] = \{([^}]*)\}", src).group(1).split(",")]
    col = [int(v) for v in re.search(r"J_COL\[\] = \{([^}]*)\}", src).group(1).split(",")]
    assert len(last) == mdl.n_terms + 1 and sum(last[:-1]) == mdl.n_couplings          # every column is closed exactly once
    assert col[:-1] == sorted(col[:-1]) and set(col[:-1]) == set(range(mdl.n_couplings))
    t0 = [int(v) for v in re.search(r"J_T0\[\] = \{([^}]*)\}", src).group(1).split(",")]
    n_inst = int(re.search(r"#define J_NINST (\d+)", src).group(1))
    assert all(-1 <= v < n_inst for v in t0[:-1])
    import copy
    with pytest.raises(binding.Tddp4Error):
        bad = copy.deepcopy(W.config(1).model)
        bad.term_coupling = [99] * bad.n_terms
        binding.jit_source(bad, 0)
    with pytest.raises(binding.Tddp4Error):            # a coupling without a term: its column would never be written
        bad = copy.deepcopy(W.config(1).model)
        bad.term_coupling = [0] * bad.n_terms
        binding.jit_source(bad, 0)
