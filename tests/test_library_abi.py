"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/gpumonty_b200.h declares; the ctypes structs have the C layout; without a GPU the product path
fails loudly instead of falling back to anything."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    txt = open(os.path.join(ROOT, "include", "gpumonty_b200.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(gm_[a-z0-9_]+)\s*\(", txt)))


def test_library_exports_every_declared_symbol():
    from paper_2602_13198_b200 import binding
    L = binding.load_library()
    names = _declared()
    assert len(names) >= 17
    for n in names:
        assert hasattr(L, n), n
    assert sorted(binding.EXPORTS + ["gm_abi_sizes"]) == names


def test_struct_layouts_match_the_c_side():
    from paper_2602_13198_b200 import binding
    L = binding.load_library()
    sz = (ctypes.c_int * 4)()
    L.gm_abi_sizes(sz)
    assert list(sz) == [ctypes.sizeof(binding.GmParams), ctypes.sizeof(binding.GmStats),
                        binding.TRACE_DTYPE.itemsize, binding.EMIT_DTYPE.itemsize]


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2602_13198_b200 import binding, workloads as wl
    p, prim = wl.config0(Ns=1e3)
    with pytest.raises(binding.GmError) as e:
        binding.GPUMonty(p)
    assert e.value.code == -3 and "no CPU path" in str(e.value)
    with pytest.raises(binding.GmError):
        binding.fp64_peak()


def test_parameter_validation_happens_before_the_device_is_touched():
    from paper_2602_13198_b200 import binding, workloads as wl
    p, _ = wl.config0(Ns=1e3)
    for key, val in (("nu_max", p["nu_min"]), ("a_spin", 1.5), ("n_nu", 0), ("w_min", -1.0), ("thetae_min", 0.1),
                     ("abi_version", 99)):
        q = dict(p)
        q[key] = val
        if key == "a_spin":
            q["metric_kind"] = 1
        with pytest.raises(binding.GmError) as e:
            binding.GPUMonty(q)
        assert e.value.code == -1, (key, str(e.value))


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2602_13198_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                for needle in ("oracle_binding", "liboracle", "import oracle", "from oracle", "oracle.hpp", "orc_"):
                    assert needle not in txt, (f, needle)
