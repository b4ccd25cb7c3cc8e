"""Host logic of the library on the CPU: the plans (instantiation, tile geometry, grid) of the register-patch Taylor kernel
(csrc/tdse_taylor_rp_plan.h) and of the persistent Runge-Kutta kernel (csrc/tdse_rk45_persist.cuh) for BASELINE.json's five
configurations and for a sweep of odd grids -- the invariants the kernels rely on.  tests/host/plans.cu is compiled with
nvcc (host code only; no device is touched)."""
import os
import shutil
import subprocess

import numpy as np
import pytest

from paper_1308_1856_b200 import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
KEYS = ["ok", "variant", "tma", "cl", "W", "H", "WT", "n_tiles", "n_items", "grid", "threads", "persist",
        "k_ok", "G", "Wc", "R", "pitch", "smem", "kreg"]


@pytest.fixture(scope="module")
def plans(tmp_path_factory):
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not found")
    exe = str(tmp_path_factory.mktemp("plans") / "plans")
    subprocess.run([nvcc, "-std=c++17", "-O1", "-gencode", "arch=compute_100a,code=sm_100a",
                    "-I" + os.path.join(ROOT, "paper_1308_1856_b200", "csrc"), "-I" + os.path.join(ROOT, "include"),
                    "-o", exe, os.path.join(ROOT, "tests", "host", "plans.cu")], check=True, capture_output=True)

    def run(cases):
        args = [str(v) for c in cases for v in c]
        out = subprocess.run([exe, *args], check=True, capture_output=True, text=True).stdout.strip().splitlines()
        assert len(out) == len(cases)
        return [dict(zip(KEYS, map(int, line.split()))) for line in out]
    return run


def cfg_case(name, persist=0):
    c = wl.config(name)
    return (c["n_r"], c["n_l"], c["fd_order"], c["batch"], c.get("order", 4) if c["propagator"] == "taylor" else 4, persist)


def test_plans_of_the_five_configurations(plans):
    p5, p1, p1s, p2, p3, p4 = plans([cfg_case("cfg5"), cfg_case("cfg1", 8), cfg_case("cfg1"), cfg_case("cfg2"),
                                     cfg_case("cfg3"), cfg_case("cfg4")])
    # CFG5 (headline): 16-row CTAs of 4 warps, TMA tiles of 128 columns, 18 tiles of 112 interior columns, a grid that is
    # a multiple of the tile count and at most two CTAs per SM; too large for the on-chip Runge-Kutta kernel
    assert (p5["ok"], p5["variant"], p5["tma"], p5["cl"], p5["W"], p5["H"], p5["n_tiles"]) == (1, 2, 1, 1, 112, 8, 18)
    assert p5["n_items"] == 18 * 256 and p5["grid"] % 18 == 0 and p5["grid"] <= 2 * 148 and p5["k_ok"] == 0
    # CFG1: eight steps per launch on the 8-point instantiation of 8 rows; one step per launch: a 16-point instantiation
    assert (p1["variant"], p1["persist"], p1["W"], p1["H"], p1["n_items"]) == (6, 8, 64, 32, 8)
    assert p1s["persist"] == 0 and p1s["variant"] in (0, 1, 2, 3, 4)
    # CFG2: clusters of 2; on chip: 143 CTAs of 28 columns x 32 rows, two points per thread (k in registers)
    assert p2["cl"] == 2 and (p2["k_ok"], p2["G"], p2["Wc"], p2["R"], p2["kreg"]) == (1, 143, 28, 32, 1)
    assert p2["smem"] <= 224 * 1024
    # CFG3 (L2-resident): clusters of 4, direct loads with the exact halo of 20 columns (TMA tiles would round it up to
    # 24); CFG4: clusters of 8; neither fits on chip
    assert (p3["cl"], p3["tma"], p3["H"], p3["W"]) == (4, 0, 20, 88) and p3["k_ok"] == 0
    assert p4["cl"] == 8 and p4["k_ok"] == 0


def test_plan_invariants_on_odd_grids(plans):
    rng = np.random.default_rng(1308)
    cases = []
    for _ in range(300):
        fd = int(rng.choice([3, 5]))
        cases.append((int(rng.integers(4, 5000)), int(rng.integers(1, 130)), fd, int(rng.integers(1, 40)),
                      int(rng.integers(1, 13)), int(rng.choice([0, 0, 4, 8, 16]))))
    for c, p in zip(cases, plans(cases)):
        n_r, n_l, fd, batch, order, persist = c
        hw = 1 if fd == 3 else 2
        if p["ok"]:
            rows = 4 * p["threads"] // 32 // (p["WT"] // (32 * (2 if p["variant"] >= 5 else 4)))
            assert rows * p["cl"] >= n_l, (c, p)
            k = max(1, p["persist"])
            assert p["persist"] in (0, persist, persist // 2, persist // 4, persist // 8), (c, p)
            if p["n_tiles"] > 1:
                assert p["H"] >= order * hw * k and p["W"] + 2 * p["H"] == p["WT"], (c, p)
                assert p["n_tiles"] * p["W"] >= n_r > (p["n_tiles"] - 1) * p["W"], (c, p)
            else:
                assert p["W"] == n_r <= p["WT"], (c, p)
            assert p["n_items"] == p["n_tiles"] * batch and 1 <= p["grid"] <= max(p["n_items"] * p["cl"], 1), (c, p)
            if p["tma"]:
                assert n_r % 8 == 0 and p["H"] % 8 == 0 and p["persist"] == 0, (c, p)
            if p["persist"]:
                assert p["cl"] == 1 and 2 * p["W"] >= p["WT"], (c, p)
            if p["variant"] >= 5:
                assert p["persist"] > 1, (c, p)
        if p["k_ok"]:
            assert batch <= 32 and p["R"] == batch * n_l and p["G"] <= 148, (c, p)
            assert p["G"] * p["Wc"] >= n_r > (p["G"] - 1) * p["Wc"], (c, p)
            assert n_r - (p["G"] - 1) * p["Wc"] >= hw or p["G"] == 1, (c, p)
            assert p["R"] * p["Wc"] <= 2048 and p["pitch"] == p["Wc"] + 2 * hw and p["smem"] <= 224 * 1024, (c, p)
            assert p["kreg"] == int(p["R"] * p["Wc"] <= 1024), (c, p)
