"""CPU-side checks of the boundary: the C-ABI library builds/loads and exports every symbol include/jipm.h
declares, the host-only entries work, and every compute entry fails loudly without a CUDA device (no CPU
fallback).  No kernel is launched here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import __graft_entry__ as ge
from paper_2606_26341_b200 import jipm, workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    if not os.path.exists(jipm.LIB_PATH):
        ge.build()
    return jipm.lib()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "jipm.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(jipm_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(lib):
    names = declared_symbols()
    assert "jipm_create" in names and "jipm_solve_batch" in names and "jipm_destroy" in names
    for nm in names:
        assert hasattr(lib, nm), nm
    assert sorted(jipm.EXPORTS) == names


def test_default_options_match_the_oracle_options(lib):
    """Both sides read the same constants; a drift would silently break parity."""
    from oracle import ipm as oipm
    o, oo = jipm.default_options(), oipm.Options()
    for f in jipm._DOUBLE_FIELDS + jipm._INT_FIELDS:
        assert getattr(o, f) == getattr(oo, f), f
    assert lib.jipm_default_options(None) == 1


def test_family_sizes_match_workloads_and_baseline_configs(lib):
    expect = {0: (74, 54, 9), 1: (392, 312, 26), 2: (1448, 1128, 60), 3: (1452, 1332, 143)}
    for cfg, (n, m, nth) in expect.items():
        d = wl.config_dims(cfg)
        assert jipm.family_sizes(d.family, d.horizon_N, d.n_agents, d.n_obstacles, d.dt) == (n, m, nth)
        assert (d.n, d.m, d.n_theta) == (n, m, nth)
    with pytest.raises(jipm.JipmError, match="error 2"):
        jipm.family_sizes(7, 10, 1, 1, 0.1)
    with pytest.raises(jipm.JipmError, match="error 2"):
        jipm.family_sizes(0, 0, 1, 1, 0.1)
    # the inequality index of a knot is packed into 8 bits with two sentinels: at most 254 obstacles per knot
    assert jipm.family_sizes(3, 4, 1, 254, 0.05)[0] == 5 * 12 + 4 * 4 + 4 * 254
    with pytest.raises(jipm.JipmError, match="error 2"):
        jipm.family_sizes(3, 4, 1, 255, 0.05)


def test_compute_entries_fail_loudly_without_a_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    d = wl.config_dims(0)
    xL, xU = wl.bounds(d)
    with pytest.raises(jipm.JipmError, match="error 4"):
        jipm.Solver(d.family, d.horizon_N, d.n_agents, d.n_obstacles, d.dt, xL, xU)
    v = C.c_double()
    assert lib.jipm_bench_fp64_peak(None, C.byref(v)) == 4
    assert b"no CUDA device" in lib.jipm_last_error()
    assert lib.jipm_solve_batch(None, 1, None, None, None, None, None, None, None, None) == 1
    assert lib.jipm_destroy(None) == 0


def test_create_argument_checks_come_before_the_device_check(lib):
    d = wl.config_dims(0)
    xL, xU = wl.bounds(d)
    h = C.c_void_p()
    dims = jipm.FamilyDims(d.horizon_N, 1, 1, d.dt)
    assert lib.jipm_create(C.byref(h), d.family, C.byref(dims), d.n + 1, d.m, xL.ctypes.data, xU.ctypes.data,
                           None, 0, None) == 2
    assert lib.jipm_create(None, d.family, C.byref(dims), d.n, d.m, xL.ctypes.data, xU.ctypes.data, None, 0, None) == 1
    assert lib.jipm_create(C.byref(h), d.family, C.byref(dims), d.n, d.m, xL.ctypes.data, xU.ctypes.data,
                           None, -1, None) == 1


def test_product_path_does_not_import_the_oracle():
    """The product path must not route through oracle/ (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2606_26341_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith(".py"):
            txt = open(os.path.join(ROOT, "oracle", fn)).read()
            assert "paper_2606_26341_b200" not in re.sub(r'""".*?"""', "", txt, flags=re.S), fn


def test_generators_are_counter_based():
    """Inputs of problem i do not depend on the batch they are generated in (bench shards by first_id)."""
    for cfg in range(4):
        d, th, x0 = wl.generate(cfg, 6)
        d2, th2, x02 = wl.generate(cfg, 3, first_id=3)
        assert np.array_equal(th[3:], th2) and np.array_equal(x0[3:], x02)
