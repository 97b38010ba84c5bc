"""dnslab_scalar_stats_static -- the entry point for callers that cannot allocate device memory -- against the
existing dnslab_scalar_stats on the same fields (include/dnslab.h has the full contract).

Who needs it: a monitoring plug-in that is handed a running solver's borrowed field pointers when the HBM is
already fully committed (a second workspace or a cudaMalloc would fail), and code that must not stall the device
or break a stream capture with an allocation.  The entry point therefore keeps its scratch in a fixed 1 MiB array
inside the library, which every call on the device shares and which keeps the previous call's contents.  That is
what these tests lean on: calls are made in pairs, back to back on one stream, the second with a different and
smaller box than the first, so stale partial sums from the first call would show up in the second result.

The file is named test_zz_* so that pytest collects it last: with `-x` a failure here must not hide other tests.
It passes alone in a fresh process (the first call does the one-time address look-up) and after the other files.
Tolerance: the one tests/test_parity_gpu.py uses for the box statistics (1e-12; the two paths sum in different,
fixed orders)."""
import ctypes as C

import numpy as np
import pytest

from paper_2204_02107_b200 import binding, cases

pytestmark = pytest.mark.gpu


def _close(got, ref):
    (mg, sg, ng), (mr, sr, nr) = got, ref
    return int(ng) == nr and abs(mg - mr) <= 1e-12 * max(abs(mr), 1e-300) + 1e-15 and abs(sg - sr) <= 1e-12 * max(sr, 1.0)


def test_static_scratch_stats_match_the_workspace_path_on_two_calls_in_a_row():
    import torch
    case = cases.duct_room(64, 32, 32)
    s = binding.solver_for_case(case)
    s.step(2)                                       # a c field with some structure next to the walls
    nz, ny, nx = case["shape"]
    # what the caller owns: its mask, two result slots (made once, up front), and a view of the solver's c
    mask = torch.from_numpy(np.ascontiguousarray(case["mask"], dtype=np.uint8)).to(s.device)
    out = torch.zeros(2, 3, dtype=torch.float64, device=s.device)
    c = s.fields()["c"]
    s.synchronize()
    boxes = [((0, 0, 0), (nx, ny, nz)),             # whole grid: 1024 rows, 16-byte loads
             ((61, 30, 29), (7, 5, 6)),             # wraps on every axis, odd start: 30 rows, the cell-by-cell walk
             ((2, 3, 1), (40, 20, 30)),             # 600 rows
             ((10, 2, 2), (1, 1, 1)),               # one cell
             ((0, 0, 0), (2, 1, ny))]               # inside the wall: no fluid cell -> zeros
    ref = {b: s.scalar_stats(*b) for b in boxes}
    assert ref[boxes[-1]] == (0.0, 0.0, 0)
    for first, second in [(0, 1), (2, 3), (1, 0), (0, 4), (4, 2)]:
        # two calls in a row on one stream, no synchronisation in between; the second reuses the scratch of the first
        binding.scalar_stats_static(c, mask, *boxes[first], out[0], stream=s.stream)
        binding.scalar_stats_static(c, mask, *boxes[second], out[1], stream=s.stream)
        s.synchronize()
        got = out.cpu().numpy()
        assert _close(got[0], ref[boxes[first]]), (boxes[first], got[0], ref[boxes[first]])
        assert _close(got[1], ref[boxes[second]]), (boxes[second], got[1], ref[boxes[second]])
    # the same call twice gives the same bits (fixed summation order), and the borrowed pointer of dnslab_fields works
    # through the raw C ABI as well
    L = binding.lib()
    lo, size = (C.c_int32 * 3)(2, 3, 1), (C.c_int32 * 3)(40, 20, 30)
    cptr = s.field_ptrs()["c"]
    for slot in (0, 1):
        rc = L.dnslab_scalar_stats_static(cptr, mask.data_ptr(), nx, ny, nz, lo, size, None, out[slot].data_ptr())
        assert rc == 0, L.dnslab_strerror(rc)
    s.synchronize()
    got = out.cpu().numpy()
    assert np.array_equal(got[0], got[1]) and _close(got[0], ref[boxes[2]])
    s.close()


def test_static_scratch_without_a_mask_and_at_its_row_limit():
    """A box with exactly DNSLAB_STATIC_MAX_ROWS rows fills the whole array and is accepted; one row more is refused
    with DNSLAB_ELIMIT and launches nothing (the result slot keeps its old contents); then a small box right after
    the full one must not see its leftovers."""
    import torch
    nz, ny, nx = 256, 256, 8
    assert ny * nz == binding.STATIC_MAX_ROWS
    rng = np.random.default_rng(20240611)
    cf = rng.standard_normal((nz, ny, nx)) + 3.0
    zero = np.zeros_like(cf)
    s = binding.Solver((nz, ny, nx), (0.1, 0.1, 0.1), 1e-3, 1e-3, 1e-3)       # no mask: all fluid
    s.set_fields(zero, zero, zero, cf)
    s.synchronize()
    c = s.fields()["c"]
    out = torch.full((2, 3), -7.0, dtype=torch.float64, device=s.device)
    full, small = ((0, 0, 0), (nx, ny, nz)), ((3, 250, 100), (5, 9, 2))
    binding.scalar_stats_static(c, None, *full, out[0], stream=s.stream)
    binding.scalar_stats_static(c, None, *small, out[1], stream=s.stream)
    s.synchronize()
    got = out.cpu().numpy()
    assert _close(got[0], s.scalar_stats(*full)) and int(got[0][2]) == nx * ny * nz
    assert _close(got[1], s.scalar_stats(*small)) and int(got[1][2]) == 5 * 9 * 2
    # a box of twice as many rows on a grid twice as tall: only the size check is under test, the field is never read
    L = binding.lib()
    lo, size = (C.c_int32 * 3)(0, 0, 0), (C.c_int32 * 3)(nx, 2 * ny, nz)
    big = torch.zeros((nz, 2 * ny, nx), dtype=torch.float64, device=s.device)
    out[1].fill_(-7.0)
    rc = L.dnslab_scalar_stats_static(big.data_ptr(), None, nx, 2 * ny, nz, lo, size, None, out[1].data_ptr())
    assert rc == -5 and b"static scratch" in L.dnslab_strerror(rc)
    with pytest.raises(binding.DnslabError, match="static scratch"):
        binding.scalar_stats_static(big, None, (0, 0, 0), (nx, 2 * ny, nz), out[1])
    torch.cuda.synchronize()
    assert out[1].cpu().tolist() == [-7.0, -7.0, -7.0]
    # bad arguments are refused before anything is launched
    assert L.dnslab_scalar_stats_static(None, None, nx, ny, nz, lo, size, None, out[1].data_ptr()) == -1
    assert L.dnslab_scalar_stats_static(big.data_ptr(), None, nx + 1, ny, nz, lo, size, None, out[1].data_ptr()) == -1
    s.close()
