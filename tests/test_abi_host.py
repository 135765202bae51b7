"""Host-side checks of the C ABI (no GPU, no compute calls): the library loads, exports every
symbol include/rt.h declares, validates networks as the header says, and fails loudly -- never
falls back to a CPU path -- when no CUDA device is present."""
import ctypes
import math
import os
import re

import numpy as np
import pytest

import rt_workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def rt():
    from paper_2103_00405_b200.build import build
    build()                       # nvcc cross-compiles without a GPU
    import paper_2103_00405_b200 as rt
    rt.lib()
    return rt


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "rt.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rt_[a-z_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(rt):
    names = _declared_functions()
    assert {"rt_create", "rt_run", "rt_ensemble", "rt_destroy"} <= set(names)
    raw = ctypes.CDLL(rt.library_path())
    for name in names:
        assert hasattr(raw, name), f"{name} declared in include/rt.h but not exported"


def test_binding_has_the_same_names(rt):
    for name in _declared_functions():
        assert hasattr(rt, name), f"binding lacks {name}"


def test_result_struct_layout(rt):
    assert rt.RESULT_DTYPE.itemsize == 24
    assert [rt.RESULT_DTYPE.fields[n][1] for n in ("t", "firings", "stop", "status")] == [0, 8, 16, 20]


def test_strerror_is_total(rt):
    for code in range(-9, 2):
        assert isinstance(rt.rt_strerror(code), str) and rt.rt_strerror(code)
    assert rt.rt_strerror(rt.RT_OK) == "ok"


def test_validate_accepts_all_workloads(rt):
    for name in ("cfg1", "cfg2"):
        net, x0, par = W.make_config(name)
        assert rt.rt_validate_network(net) == rt.RT_OK
    for name in ("cfg3", "cfg4"):
        net, x0, par = W.make_config(name, scale=0.01)
        assert rt.rt_validate_network(net) == rt.RT_OK


def _lv():
    net, _ = W.lotka_volterra()
    return {k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in net.items()}


@pytest.mark.parametrize("mutate,code", [
    (lambda n: n.__setitem__("n_species", 0), "RT_ERR_BAD_NETWORK"),
    (lambda n: n["react_ptr"].__setitem__(0, 1), "RT_ERR_BAD_NETWORK"),
    (lambda n: n["react_ptr"].__setitem__(1, 5), "RT_ERR_BAD_NETWORK"),          # decreasing later
    (lambda n: n["react_species"].__setitem__(0, 7), "RT_ERR_BAD_NETWORK"),      # species out of range
    (lambda n: n["react_sigma"].__setitem__(0, 0), "RT_ERR_BAD_NETWORK"),        # sigma < 1
    (lambda n: n["react_sigma"].__setitem__(0, 4), "RT_ERR_UNSUPPORTED"),        # sigma > 3
    (lambda n: n["stoich_v"].__setitem__(0, 0), "RT_ERR_BAD_NETWORK"),           # v = 0 entry
    (lambda n: n["stoich_v"].__setitem__(len(n["stoich_v"]) - 1, -3), "RT_ERR_BAD_NETWORK"),  # v < -sigma
    (lambda n: n["rate"].__setitem__(1, -1.0), "RT_ERR_BAD_NETWORK"),
    (lambda n: n["rate"].__setitem__(1, math.nan), "RT_ERR_BAD_NETWORK"),
    (lambda n: n["rate"].__setitem__(1, math.inf), "RT_ERR_BAD_NETWORK"),
])
def test_validate_rejects(rt, mutate, code):
    net = _lv()
    mutate(net)
    assert rt.rt_validate_network(net) == getattr(rt, code)


def test_validate_rejects_duplicate_species_in_a_row(rt):
    """A + A must be written sigma = 2, not two sigma = 1 entries (reading G18)."""
    net = W.from_reactions(2, [({0: 2}, {1: 1}, 1.0)])
    assert rt.rt_validate_network(net) == rt.RT_OK
    net["react_ptr"] = np.array([0, 2], dtype=np.int64)
    net["react_species"] = np.array([0, 0], dtype=np.int32)
    net["react_sigma"] = np.array([1, 1], dtype=np.int32)
    assert rt.rt_validate_network(net) == rt.RT_ERR_BAD_NETWORK


def test_no_cpu_fallback_without_a_device(rt):
    """On a machine without a GPU rt_create must fail with RT_ERR_CUDA (never simulate on the host)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    net, x0 = W.lotka_volterra()
    rc, handle = rt.rt_create(net, 0)
    assert rc == rt.RT_ERR_CUDA and handle is None
    with pytest.raises(rt.RtError):
        rt.Model(net)


def test_destroy_null_is_noop(rt):
    rt.rt_destroy(None)
    rt.rt_destroy(0)


def test_product_path_never_imports_the_oracle():
    """The package and bench's CUDA arm must not route through oracle/ (only tests, smoke and the
    cpu_baseline / --impl reference legs may)."""
    pkg = os.path.join(ROOT, "paper_2103_00405_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "rt_oracle" not in text, f
