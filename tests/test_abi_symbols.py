"""CPU: the C-ABI library builds, loads, and exports every function include/*.h declares."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared(headers=None):
    inc = os.path.join(ROOT, "include")
    names = set()
    for h in headers or sorted(f for f in os.listdir(inc) if f.endswith(".h")):
        src = open(os.path.join(inc, h)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names |= set(re.findall(r"\b(pimd_[a-z_]+)\s*\(", src))
    return sorted(names)


def test_header_declares_the_north_star_calls():
    names = _declared(["pimd.h"])
    assert not any(n.startswith("pimd_debug") or n == "pimd_time_kernel" for n in names)    # hooks live in pimd_debug.h
    for need in ["pimd_create", "pimd_set_model", "pimd_step", "pimd_get_positions", "pimd_get_momenta",
                 "pimd_get_forces", "pimd_get_virial", "pimd_get_estimators", "pimd_destroy"]:
        assert need in names


def test_library_builds_and_exports_every_declared_symbol():
    import __graft_entry__ as ge
    ge.build()
    import ctypes
    import paper_2602_13553_b200 as pk
    L = ctypes.CDLL(pk.library_path())
    for name in _declared():
        assert hasattr(L, name), name
    # the binding binds the same names
    for name in _declared():
        assert hasattr(pk, name), name


def test_no_cpu_fallback_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    import numpy as np
    import paper_2602_13553_b200 as pk
    with pytest.raises(pk.PimdError) as ei:
        pk.pimd_create(np.zeros(3, np.int32), [1.0], [10.0, 10.0, 10.0], 4, 300.0, 1e-3, 1.0, 0)
    assert ei.value.code == pk.PIMD_ECUDA


def test_model_weight_count_matches_workload_generator():
    import paper_2602_13553_b200 as pk
    import workloads
    desc = workloads.model_desc()
    assert pk.pimd_model_n_weights(pk.ModelDesc.from_dict(desc)) == workloads.n_model_weights(desc) == 1026122


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2602_13553_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
