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


def test_scalar_stats_static_validates_before_touching_the_device(L):
    """The entry point that allocates nothing checks its arguments -- and the row limit of its static scratch array --
    before any CUDA call, so the refusals can be seen without a GPU; the pointers below are never dereferenced."""
    fake = 0x1000
    lo, size = (C.c_int32 * 3)(0, 0, 0), (C.c_int32 * 3)(8, 8, 8)
    f = L.dnslab_scalar_stats_static
    assert f(None, None, 8, 8, 8, lo, size, None, fake) == -1                     # no c
    assert f(fake, None, 8, 8, 8, lo, size, None, None) == -1                     # no out
    assert f(fake, None, 8, 12, 8, lo, size, None, fake) == -1                    # ny not a power of two
    assert f(fake, None, 4096, 8, 8, lo, size, None, fake) == -1                  # nx beyond the library's grids
    assert f(fake, None, 8, 8, 8, lo, (C.c_int32 * 3)(9, 1, 1), None, fake) == -1  # box wider than the grid
    assert f(fake, None, 8, 8, 8, lo, (C.c_int32 * 3)(1, 0, 1), None, fake) == -1
    big = (C.c_int32 * 3)(8, 512, 256)                                            # 131 072 rows > DNSLAB_STATIC_MAX_ROWS
    assert binding.STATIC_MAX_ROWS == 65536
    assert f(fake, None, 8, 512, 256, lo, big, None, fake) == -5
    assert b"static scratch" in L.dnslab_strerror(-5)
    import torch
    if not torch.cuda.is_available():
        ok = (C.c_int32 * 3)(8, 256, 256)                                         # exactly the limit: passes the checks, then no device
        assert f(fake, None, 8, 256, 256, lo, ok, None, fake) == -4


def test_bench_traffic_lookup_and_workload_string():
    """bench.py host logic: roofline.traffic comes from the committed ncu export of the line's own workload, is None
    (not an exception) for an export with an unknown unit or of another workload, and both arms name the workload alike."""
    import argparse
    import sys
    import tempfile
    sys.path.insert(0, ROOT)
    import bench
    from paper_2204_02107_b200 import cases
    a = argparse.Namespace(config=4, mode="step", traffic_csv=None)
    t, src = bench.ncu_traffic(bench.default_traffic_csv(a), "rk_stage", {"name": "room512x256x128"})
    assert t is not None and 1.5e9 < t < 1.7e9, (t, src)                          # 96 B/cell x 16.8 M cells
    assert bench.ncu_traffic(bench.default_traffic_csv(a), "rk_stage", {"name": "duct128x64x64"})[0] is None
    assert bench.default_traffic_csv(argparse.Namespace(config=2, mode="step", traffic_csv=None)) is None
    for cfg, mode, cls, name in [(3, "step", "rk_stage", "turb256"), (5, "step", "rk_stage", "rooms1024x512x256"),
                                 (4, "reductions", "k_courant", "room512x256x128"), (4, "particles", "particles", "room512x256x128")]:
        a = argparse.Namespace(config=cfg, mode=mode, traffic_csv=None)
        assert bench.ncu_traffic(bench.default_traffic_csv(a), cls, {"name": name})[0] is not None, (cfg, mode)
    with tempfile.TemporaryDirectory() as d:
        p = os.path.join(d, "x.csv")
        with open(p, "w") as fh:
            fh.write('"Kernel Name","dram__bytes_read.sum","dram__bytes_write.sum"\n"","Pbyte","Pbyte"\n"k_rk_march<1>","1","1"\n')
        with open(os.path.join(d, "x.md"), "w") as fh:
            fh.write("room512x256x128")
        t, src = bench.ncu_traffic(p, "rk_stage", {"name": "room512x256x128"})
        assert t is None and "unknown unit" in src
    case = cases.config(2)
    w = bench.workload_name(2, case)
    assert w.startswith("config 2: duct128x64x64 (524288 cells), n_piter=4")
