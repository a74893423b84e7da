"""Host-side checks that need no GPU: the library builds/loads, exports every symbol include/lbm.h declares,
and its argument validation answers with the documented codes."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2607_04516_b200 import build, binding
    build.build()
    return binding.load_library()


def _declared():
    text = open(os.path.join(ROOT, "include", "lbm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lbm_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    from paper_2607_04516_b200 import binding
    names = _declared()
    assert len(names) >= 25
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/lbm.h but not exported"
    assert sorted(binding.SYMBOLS) == names


def test_workspace_bytes_counts_two_buffers_flags_and_mean(lib):
    out = C.c_size_t()
    assert lib.lbm_workspace_bytes(400, 400, 100, 0, 0, C.byref(out)) == 0
    # halo-padded box: x pitch = nx + 2 rounded up to 32, one halo layer in y and z
    n = 416 * 402 * 102  # 400 + 8 (row offset) + 1 (halo) -> 416
    per_cell = 2 * 19 * 4 + 1 + 4  # two population buffers, flag byte, link word
    assert out.value >= per_cell * n
    assert out.value < per_cell * n + 32 * 2 ** 20   # side arrays: face velocities (two halves + mean), mode table, damping tables, scratch
    with_mean = C.c_size_t()
    assert lib.lbm_workspace_bytes(400, 400, 100, 1, 0, C.byref(with_mean)) == 0
    assert with_mean.value - out.value == pytest.approx(12 * n, rel=1e-3)
    f64 = C.c_size_t()
    assert lib.lbm_workspace_bytes(400, 400, 100, 0, 1, C.byref(f64)) == 0
    assert f64.value >= 2 * 19 * 8 * n
    assert lib.lbm_workspace_bytes(0, 4, 4, 0, 0, C.byref(out)) == -1
    assert lib.lbm_workspace_bytes(4, 4, 4, 0, 0, None) == -1
    assert lib.lbm_workspace_bytes(2000, 2000, 2000, 0, 0, C.byref(out)) == -1  # beyond int32 cell indices


def test_null_handle_and_bad_arguments_return_codes(lib):
    assert lib.lbm_step(None, 1) == -1
    assert lib.lbm_destroy(None) == -1
    assert lib.lbm_get_step(None) == -1
    assert lib.lbm_sync(None) == -1
    assert lib.lbm_set_flags(None, None) == -1
    assert lib.lbm_last_error(None) == b"NULL handle"
    h = C.c_void_p()
    F = (C.c_double * 3)(0, 0, 0)
    assert lib.lbm_create(0, 4, 4, 1e-3, 0.1, 0.0, F, C.byref(h)) == -1
    assert lib.lbm_create(4, 4, 4, -1.0, 0.1, 0.0, F, C.byref(h)) == -1
    assert lib.lbm_create(4, 4, 4, 1e-3, 0.1, 0.0, F, None) == -1


def test_create_without_a_device_fails_loudly(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    h = C.c_void_p()
    F = (C.c_double * 3)(0, 0, 0)
    assert lib.lbm_create(4, 4, 4, 1e-3, 0.1, 0.0, F, C.byref(h)) == -3  # LBM_ECUDA: no CPU fallback
    from paper_2607_04516_b200 import binding
    with pytest.raises(binding.LbmError):
        binding.Lbm(4, 4, 4, 1e-3)


def test_library_lattice_matches_the_documented_order(lib):
    from paper_2607_04516_b200 import binding
    c, opp = binding.lattice()
    firsts = [(1, 0, 0), (0, 1, 0), (0, 0, 1), (1, 1, 0), (1, 0, 1), (0, 1, 1), (1, -1, 0), (1, 0, -1), (0, 1, -1)]
    assert tuple(c[0]) == (0, 0, 0) and opp[0] == 0
    for k, v in enumerate(firsts):
        assert tuple(c[2 * k + 1]) == v and tuple(c[2 * k + 2]) == tuple(-a for a in v)
        assert opp[2 * k + 1] == 2 * k + 2 and opp[2 * k + 2] == 2 * k + 1


def test_product_package_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2607_04516_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "lbm_oracle" not in src, f


def test_workloads_match_the_config_statements():
    from paper_2607_04516_b200 import workloads as W
    c1 = W.config1()
    assert (c1.nx, c1.ny, c1.nz) == (64, 32, 32) and c1.height.sum() == 8 * 8 * 16
    assert c1.inlet_profile[0][15] == pytest.approx(0.05 * np.log(15.5 / 0.1) / np.log(160), rel=1e-6)
    c3 = W.config3()
    hm = c3.height
    assert hm.shape == (400, 400) and hm.max() <= 40 and (hm[:, :8] == 0).all() and (hm[:, -8:] == 0).all()
    assert 0.35 <= (hm > 0).mean() < 0.36
    assert np.array_equal(hm, W.config3().height)  # seeded
    u = c3.inlet_profile[0]
    assert u[19] < 0.08 < u[20] or u[19] == pytest.approx(0.08, rel=0.02)
    c2 = W.config2()
    assert c2.init[1].shape == (128, 128, 128) and abs(float(c2.init[1].mean()) - 0.02) < 1e-6
