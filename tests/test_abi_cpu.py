"""CPU-side checks of the product library: it builds for sm_100a, loads without a GPU, exports every symbol that
include/tdse.h declares, and refuses to compute without a CUDA device (there is no CPU fallback)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_1308_1856_b200 import build
    build.build()
    from paper_1308_1856_b200 import binding as b
    return b


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "tdse.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(tdse_[a-zA-Z0-9_]+)\s*\(", text)))


def test_header_symbols_exported(binding):
    names = declared_symbols()
    assert len(names) >= 18
    lib = binding.lib()
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(binding.SYMBOLS) == names            # the binding wraps exactly what the header declares
    assert binding.version().startswith("tdse_b200")
    assert binding.strerror(-5) == "unsupported configuration"


def test_struct_layouts_match_header(binding):
    assert C.sizeof(binding.Grid) == 48 and C.sizeof(binding.Pulse) == 40      # 4 doubles + int kind (padded)
    assert binding.Grid.dr.offset == 8 and binding.Grid.z_nuc.offset == 32 and binding.Grid.batch.offset == 40


def test_no_cpu_fallback(binding):
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    with pytest.raises(binding.TdseError) as ei:
        binding.Tdse(100, 0.2, 3, 3)
    assert ei.value.code == -3                          # TDSE_ERR_CUDA: fails loudly, computes nothing
    hp = C.c_void_p()
    assert binding.lib().tdse_create(None, C.byref(hp)) == -1
    assert binding.lib().tdse_launch_count(None) == 0


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1308_1856_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "tdse_oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "binding" not in src and "libtdse_b200" not in src and "csrc" not in src.replace("csrc/,", ""), f


def test_bench_bound_state_inputs_match_the_oracle():
    """bench.py's product arm may not touch oracle/, so it takes CFG5's bound states (every E < 0 eigenvector of the
    discrete 3-point h_l) from LAPACK; they must be the same input data the GPU tests take from the oracle's eigen-solver."""
    import numpy as np
    import oracle
    import bench
    from paper_1308_1856_b200 import workloads as wl
    c = wl.config("cfg5", n_r=400, n_l=4, batch=1)
    ls, phis = bench.bound_state_inputs(c)
    g = oracle.make_grid(c["n_r"], c["dr"], c["n_l"], 3)
    k = 0
    for l in range(c["n_l"]):
        en, phi = oracle.bound_states(g, l, 32, only_negative=True)
        assert list(ls[k:k + len(en)]) == [l] * len(en)
        for i in range(len(en)):
            assert abs(c["dr"] * np.sum(phis[k + i] ** 2) - 1.0) < 1e-12 and phis[k + i][0] > 0
            assert np.max(np.abs(phis[k + i] - phi[i])) < 1e-8
        k += len(en)
    assert k == len(ls) and k >= 6
