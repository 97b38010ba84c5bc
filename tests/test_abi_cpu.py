"""CPU-side checks of the C ABI: the library loads without a GPU, exports every symbol that
include/dnslab.h declares, and validates parameters (no compute calls here)."""
import ctypes as C
import os
import re

import pytest

from paper_2204_02107_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    build.build()
    return binding.lib()


def test_every_declared_symbol_is_exported(L):
    hdr = open(os.path.join(ROOT, "include", "dnslab.h")).read()
    declared = set(re.findall(r"\b(dnslab_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(binding.SYMBOLS)
    for name in declared:
        assert hasattr(L, name), name


def test_struct_layout_matches_header():
    assert C.sizeof(binding.Params) == 96
    assert C.sizeof(binding.Source) == 96


def test_workspace_bytes_validates(L):
    ok = binding.make_params((16, 32, 64), (0.1, 0.1, 0.1), 1e-3, 1e-3, 1e-2, n_piter=4)
    n = 16 * 32 * 64
    w = binding.workspace_bytes(ok)
    assert w >= 19 * 8 * n + n and w % 256 == 0
    assert binding.workspace_bytes(binding.make_params((16, 32, 64), (0.1, 0.1, 0.1), 1e-3, 1e-3, 1e-2, flags=2)) >= w + 8 * n
    bad = [dict(shape=(16, 32, 48)), dict(shape=(4, 32, 64)), dict(shape=(16, 2048, 64)), dict(shape=(16, 32, 4096)),
           dict(d=(0.0, 0.1, 0.1)), dict(dt=0.0), dict(nu=-1.0), dict(n_piter=0), dict(flags=4), dict(flags=8), dict(flags=16),
           dict(dt=float("nan"))]
    for b in bad:
        kw = dict(shape=(16, 32, 64), d=(0.1, 0.1, 0.1), nu=1e-3, alpha_c=1e-3, dt=1e-2, n_piter=1, flags=0)
        kw.update(b)
        assert binding.workspace_bytes(binding.make_params(**kw)) == 0, b


def test_null_handle_and_strerror(L):
    assert L.dnslab_step(None, 1) == -1
    assert L.dnslab_destroy(None) == -1
    assert L.dnslab_launch_count(None) == -1
    assert L.dnslab_strerror(0) == b"ok"
    assert b"workspace" in L.dnslab_strerror(-2)
    assert L.dnslab_strerror(-99) == b"unknown error"


def test_no_gpu_means_loud_failure():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(binding.DnslabError):
        binding.Solver((8, 8, 8), (1.0, 1.0, 1.0), 0.1, 0.1, 0.1)


def test_product_path_never_touches_the_oracle():
    pkg = os.path.join(ROOT, "paper_2204_02107_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "dnsref" not in txt and "import oracle" not in txt and "from oracle" not in txt, f
    for f in ("dnsref.c", "dnsref.py"):
        txt = open(os.path.join(ROOT, "oracle", f)).read()
        assert "libdnslab" not in txt and "binding" not in txt and "csrc/" not in txt.replace("paper_2204_02107_b200/csrc/", "")
