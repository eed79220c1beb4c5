"""CPU-side checks of the boundary: the CUDA library builds (nvcc cross-compiles), loads without a GPU, and exports
every symbol include/pt.h declares; the binding refuses host tensors (there is no CPU fallback)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "pt.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(?:int|int64_t)\s+(pt_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def libpath():
    from paper_1504_07433_b200 import build
    return build.build()


def test_header_declares_the_north_star_entry_points():
    names = declared_functions()
    for n in ("pt_orbit_z", "pt_ma_quad_exact", "pt_ma_table_build", "pt_ma_quad_interp"):
        assert n in names


def test_library_exports_every_declared_symbol(libpath):
    L = ctypes.CDLL(libpath)
    for n in declared_functions():
        assert hasattr(L, n), n
    L.pt_build_arch.restype = ctypes.c_int
    assert L.pt_build_arch() == 100
    L.pt_launch_count.restype = ctypes.c_int64
    assert L.pt_launch_count() == 0


def test_binding_matches_header_and_has_no_cpu_path(libpath):
    import torch
    import paper_1504_07433_b200 as pt
    from paper_1504_07433_b200 import binding
    assert sorted(binding.EXPORTS) == declared_functions()
    for n in binding.EXPORTS:
        assert hasattr(binding.lib(), n)
    t = torch.zeros(4, dtype=torch.float64)
    p = torch.zeros((1, 9), dtype=torch.float64)
    with pytest.raises(binding.PtError):
        pt.pt_ma_quad_exact(t, p)
    with pytest.raises(binding.PtError):
        pt.pt_orbit_z(t, p)
    with pytest.raises(binding.PtError):
        pt.pt_ma_quad_exact(t.float(), p)
    # argument validation happens before any CUDA call, so it can be exercised without a GPU
    L = binding.lib()
    buf = (ctypes.c_double * 16)()
    a = ctypes.addressof(buf)
    assert L.pt_ma_quad_exact(None, 4, 0, a, 1, 1, 1, 0.0, 0, a, None, None) == binding.PT_ERR_NULL
    assert L.pt_ma_quad_exact(a, -1, 0, a, 1, 1, 1, 0.0, 0, a, None, None) == binding.PT_ERR_SIZE
    assert L.pt_orbit_z(a, 4, 2, a, 1, 1, 1, 0.0, a, None) == binding.PT_ERR_SIZE
    assert L.pt_ma_table_build(0.1, 0.2, 1, 1.2, 10, 0, 3, a, None) == binding.PT_ERR_SIZE
    assert L.pt_ma_table_build(0.1, 0.2, 4, 1.2, 10, 5, 3, a, None) == binding.PT_ERR_DTYPE


def test_missing_extension_fails_loudly(monkeypatch, tmp_path):
    from paper_1504_07433_b200 import binding
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(binding.PtError, match="no CPU fallback"):
        binding.lib()


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1504_07433_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "pt_oracle" not in txt and "ma_definition" not in txt and "from oracle" not in txt, f
    for f in ("pt_oracle.cpp", "pt_oracle.py", "ma_definition.py"):
        txt = open(os.path.join(ROOT, "oracle", f)).read()
        assert "paper_1504_07433_b200" not in txt.replace("paper_1504_07433_b200/csrc/", ""), f


def test_input_generators_are_seeded_and_shaped():
    from paper_1504_07433_b200 import inputs
    a, b = inputs.config2(), inputs.config2()
    assert np.array_equal(a.times, b.times) and np.array_equal(a.params, b.params)
    assert a.params.shape == (64, 9) and a.times.shape == (60000,) and a.n_ss == 10 and a.n_eval == 38400000
    assert not np.array_equal(a.params, inputs.config2(stream=1).params)
    c = inputs.config3()
    assert c.params.shape == (512, 66) and c.times.shape == (600,) and c.n_pb == 20
    d = inputs.config4(n_pv=16, n_t=100)
    assert d.table == dict(k_min=0.05, k_max=0.25, n_k=401, z_max=1.25, n_z=12501)
    assert inputs.config1().times.shape == (1000,)
    k = a.params[:, 6]
    assert k.min() >= 0.05 and k.max() <= 0.2
    u1, u2 = a.params[:, 7], a.params[:, 8]
    assert np.all(u1 + u2 <= 1 + 1e-12) and np.all(u1 >= 0) and np.all(u1 + 2 * u2 >= -1e-12)   # Kipping's triangle


def test_launch_plan_host_logic(libpath):
    """Tiling / scheduling decisions of the host side (pt_plan: no CUDA call), for the five BASELINE shapes on 148 SMs."""
    from paper_1504_07433_b200 import binding
    warps = 148 * 3 * 8
    # configs[1]: 64 rows of 60000 -> few rows, many tiles per warp: longest-processing-time-first order, full grid
    p = binding.pt_plan(64, 60000)
    assert p["mode"] == 2 and p["tile_len"] % 256 == 0 and p["blocks"] == 148 * 3
    assert p["tiles_per_pv"] == -(-60000 // p["tile_len"]) and 64 * p["tiles_per_pv"] >= 2 * warps
    # configs[0]: one short row -> a latency: short tiles, one round of many warps
    p = binding.pt_plan(1, 1000)
    assert p["mode"] in (0, 1) and p["tile_len"] == 32 and p["blocks"] == 4 and p["tile_len"] * p["tiles_per_pv"] >= 1000
    # configs[2]: 512 rows of 600 -> fewer tiles than warps: no ranking, per-row counters
    p = binding.pt_plan(512, 600)
    assert p["mode"] == 1 and p["tiles_per_pv"] == 3
    # configs[3]: 4096 rows of 100000 -> too many rows for per-row counters: global counter, long tiles, full grid
    p = binding.pt_plan(4096, 100000)
    assert p["mode"] == 0 and p["tile_len"] == 14592 and p["tiles_per_pv"] == 7 and p["blocks"] == 148 * 3
    # configs[4]: 4096 rows of 4096
    p = binding.pt_plan(4096, 4096)
    assert p["mode"] == 0 and p["tile_len"] * p["tiles_per_pv"] >= 4096 and p["blocks"] == 148 * 3
    # every exposure is covered exactly once whatever the shape; the grid never exceeds three blocks per SM
    for n_pv, n_t, n_sm in ((1, 1, 148), (3, 255, 148), (3, 257, 132), (1000, 7, 148), (7, 10 ** 7, 148), (10 ** 6, 3, 148),
                            (448, 60000, 148), (2, 2 ** 31 - 1, 8)):
        p = binding.pt_plan(n_pv, n_t, n_sm)
        assert 32 <= p["tile_len"] <= 16384 and p["tile_len"] % 32 == 0
        assert p["tile_len"] % 256 == 0 or n_pv * n_t < 64 * n_sm              # short tiles only for tiny problems
        assert (p["tiles_per_pv"] - 1) * p["tile_len"] < n_t <= p["tiles_per_pv"] * p["tile_len"]
        assert 1 <= p["blocks"] <= n_sm * 3
    with pytest.raises(binding.PtError):
        binding.pt_plan(0, 10)
