"""CPU-only checks of the boundary: libmdg.so builds, loads, exports every symbol include/mdg.h
declares, the ctypes mirror of mdg_params matches, and without a GPU the library fails loudly."""
import ctypes as C
import os
import re

import pytest

import paper_2606_08039_b200 as mdg
from paper_2606_08039_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return mdg.lib()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "mdg.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mdg_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    syms = declared_symbols()
    assert len(syms) >= 18 and "mdg_step" in syms and "mdg_step_host" in syms
    for s in syms:
        assert hasattr(lib, s), f"libmdg.so does not export {s}"
    assert set(binding.EXPORTS) <= set(syms)


def test_params_struct_mirror_and_defaults(lib):
    p = mdg.default_params()
    assert p.struct_size == C.sizeof(mdg.mdg_params)
    # Table 2, Table 6
    assert abs(p.m / 0.027 - 1) < 1e-6 and abs(p.L / 0.0397 - 1) < 1e-6 and abs(p.tw_ratio - 2.25) < 1e-6
    assert abs(p.k_f / 3.16e-10 - 1) < 1e-6 and abs(p.k_m / 7.94e-12 - 1) < 1e-6
    assert all(abs(a / b - 1) < 1e-6 for a, b in zip(p.J, [1.4e-5, 1.4e-5, 2.17e-5]))
    assert [round(x, 6) for x in p.Kp_pos] == [0.4, 0.4, 1.0] and [round(x, 6) for x in p.Kd_pos] == [0.9, 0.9, 2.0]
    assert (round(p.dw_C1, 2), round(p.dw_C2, 2), round(p.dw_C3, 2)) == (2267.18, 0.16, -0.11)
    assert (p.sim_freq, p.ctrl_freq) == (240, 48) and p.env_index_base == 0
    race = mdg.default_params(2)
    assert abs(race.m - 0.25) < 1e-6 and abs(race.tw_ratio - 4.0) < 1e-6
    with pytest.raises(mdg.MdgError):
        mdg.default_params(7)
    with pytest.raises(AttributeError):
        mdg.default_params(0, no_such_field=1)


def test_argument_validation_and_no_cpu_fallback(lib):
    import torch
    h = C.c_void_p()
    p = mdg.default_params()
    assert lib.mdg_create(0, 1, 0, 0, C.byref(p), C.byref(h)) == binding.MDG_EINVAL
    assert lib.mdg_create(4, 33, 0, 0, C.byref(p), C.byref(h)) == binding.MDG_EINVAL
    assert lib.mdg_create(4, 1, 9, 0, C.byref(p), C.byref(h)) == binding.MDG_EINVAL
    bad = mdg.default_params(0, sim_freq=250)
    assert lib.mdg_create(4, 1, 0, 0, C.byref(bad), C.byref(h)) == binding.MDG_EINVAL
    assert b"multiple of ctrl_freq" in lib.mdg_last_error()
    bad = mdg.default_params()
    bad.struct_size = 12
    assert lib.mdg_create(4, 1, 0, 0, C.byref(bad), C.byref(h)) == binding.MDG_EINVAL
    if not torch.cuda.is_available():
        assert lib.mdg_create(4, 1, 0, 0, C.byref(p), C.byref(h)) == binding.MDG_ECUDA
        assert b"no CPU fallback" in lib.mdg_last_error()
        with pytest.raises(RuntimeError):
            mdg.Env(4, 1, 0, 0)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_08039_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.lower() or f in ("workloads.py", "mdg_dev.cuh", "__init__.py"), f
    for f in ("drone_oracle.hpp", "camera_oracle.hpp", "oracle_capi.cpp", "philox_ref.hpp", "oracle.py"):
        txt = open(os.path.join(ROOT, "oracle", f)).read()
        assert "paper_2606_08039_b200" not in txt.replace("paper_2606_08039_b200/csrc", "") and "mdg.h\"" not in txt
