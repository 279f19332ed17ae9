"""ecsim_cell_segments_static: the per-cell counts and segment table of a species for callers that cannot allocate.

Why the entry point exists.  Every other libecpush call wants a context (events, pinned host buffers) and a workspace
that the caller got from cudaMalloc.  A caller that lives inside somebody else's memory plan cannot provide one: a
plug-in called from a host code whose device memory is given out once at start-up (ECsim's OpenACC data regions, a
framework pool that already owns the whole HBM), or a time loop that cannot afford the device-wide stall of cudaMalloc
/ cudaFree.  For them the histogram and the scan's partial sums sit in an 8 MB array that is part of libecpush.so's
device image (grids up to ECSIM_STATIC_MAX_CELLS = 128^3 cells); the caller passes only its inputs and outputs.

What is checked.  The array is shared by all calls and keeps the previous call's contents, so a call that forgot to
clear the histogram would be right once and wrong the second time.  The GPU test therefore makes two calls in a row,
without a synchronisation between them, on DIFFERENT species and grids (the second grid smaller, so stale counts of
the first would lie inside and beyond it), then the first again, and compares every result with the existing path --
ecsim_sort_particles of a context with a lent workspace -- bit for bit (integer work: the repo's tolerance for cell ids
and counts is equality).  The file is named test_zz_* so that pytest collects it after every other test file: with
`pytest -x` a failure here cannot hide the parity tests.  It holds no state of its own and needs none from other
tests, so it passes alone in a fresh process as well as at the end of the whole run.
"""
from __future__ import annotations

import re

import numpy as np
import pytest
import torch

import paper_2603_16624_b200 as pk
from paper_2603_16624_b200 import binding
from util import PKEYS, rand_particles


def _counts_by_existing_path(grid, pn):
    """Per-cell counts from the context-based path: ecsim_sort_particles with a workspace lent by torch."""
    n = pn["x"].size
    cells = grid[0] * grid[1] * grid[2]
    ctx = pk.Ecsim(*grid, 1)
    ctx.set_workspace(n)
    pc = {k: torch.from_numpy(pn[k]).cuda() for k in PKEYS}     # sorted in place: a private copy
    ctx.load_particles(0, -1.0, pc, sorted=False)
    count = torch.full((cells,), -7, dtype=torch.int32, device="cuda")
    ctx.sort_particles(0, count, None)
    torch.cuda.synchronize()
    out = count.cpu().numpy().copy()
    ctx.close()
    return out


def _static_call(grid, xyz):
    """One ecsim_cell_segments_static call; outputs pre-filled with garbage, nothing synchronised here."""
    cells = grid[0] * grid[1] * grid[2]
    count = torch.full((cells,), -5, dtype=torch.int32, device="cuda")
    start = torch.full((cells + 1,), -3, dtype=torch.int32, device="cuda")
    pk.cell_segments_static(*grid, *xyz, cell_count_out=count, start_out=start)
    return count, start


def _expect_start(count_ref):
    return np.concatenate([[0], np.cumsum(count_ref.astype(np.int64))])


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_workspace_path():
    rng = np.random.default_rng(20260316)
    # A: several scan blocks (30 * 37 * 11 = 12 210 cells > 11 x 1024) with a ragged last one, ragged particle count
    grid_a = (30, 37, 11, 0.5, 1.25, 2.0)
    pa = rand_particles(rng, 200_003, grid_a)
    # B: a smaller grid and fewer particles, clustered in a corner so that most cells are empty
    grid_b = (9, 6, 14, 0.3, 0.7, 1.1)
    pb = rand_particles(rng, 31_001, grid_b)
    pb["x"] *= 0.25
    pb["y"] *= 0.5
    ref_a = _counts_by_existing_path(grid_a, pa)
    ref_b = _counts_by_existing_path(grid_b, pb)
    assert ref_a.sum() == pa["x"].size and ref_b.sum() == pb["x"].size

    xa = [torch.from_numpy(pa[k]).cuda() for k in "xyz"]
    xb = [torch.from_numpy(pb[k]).cuda() for k in "xyz"]
    ca1, sa1 = _static_call(grid_a, xa)        # first call on this device in a fresh process: does the set-up
    cb, sb = _static_call(grid_b, xb)          # second call straight after it, same stream: sees A's leftovers
    ca2, sa2 = _static_call(grid_a, xa)        # and A once more after B
    torch.cuda.synchronize()
    for what, c, s, ref in (("A, first call", ca1, sa1, ref_a), ("B, second call", cb, sb, ref_b),
                            ("A, third call", ca2, sa2, ref_a)):
        assert np.array_equal(c.cpu().numpy(), ref), f"{what}: per-cell counts differ from ecsim_sort_particles"
        got = s.cpu().numpy().astype(np.int64) & 0xFFFFFFFF
        assert np.array_equal(got, _expect_start(ref)), f"{what}: segment table is not the running sum of the counts"
    # the inputs are read only
    for t, k in zip(xa, "xyz"):
        assert np.array_equal(t.cpu().numpy(), pa[k])


@pytest.mark.gpu
def test_single_outputs_and_empty_species():
    rng = np.random.default_rng(7)
    grid = (5, 4, 3, 1.0, 1.0, 1.0)
    cells = 60
    p = rand_particles(rng, 999, grid)
    ref = _counts_by_existing_path(grid, p)
    xyz = [torch.from_numpy(p[k]).cuda() for k in "xyz"]
    count = torch.full((cells,), -5, dtype=torch.int32, device="cuda")
    start = torch.full((cells + 1,), -3, dtype=torch.int32, device="cuda")
    pk.cell_segments_static(*grid, *xyz, cell_count_out=count)            # counts only
    pk.cell_segments_static(*grid, *xyz, start_out=start)                 # table only
    torch.cuda.synchronize()
    assert np.array_equal(count.cpu().numpy(), ref)
    assert np.array_equal(start.cpu().numpy(), _expect_start(ref))
    # no particles: every count and every start is zero, whatever the last call left in the scratch
    empty = [torch.empty(0, dtype=torch.float64, device="cuda") for _ in range(3)]
    pk.cell_segments_static(*grid, *empty, cell_count_out=count, start_out=start)
    torch.cuda.synchronize()
    assert not count.cpu().numpy().any() and not start.cpu().numpy().any()


def test_grids_beyond_the_built_in_scratch_are_refused():
    """Argument checks come before any CUDA call, so this runs on a box without a GPU too: a grid of more than
    ECSIM_STATIC_MAX_CELLS cells is an error whose text names the limit, and nothing is enqueued."""
    L = pk.lib()
    header = open(binding.HEADER).read()
    limit = int(re.search(r"#define\s+ECSIM_STATIC_MAX_CELLS\s+(\d+)", header).group(1))
    assert limit == pk.STATIC_MAX_CELLS == 128 ** 3
    one = 1 << 20                              # never dereferenced: the call returns before touching the device
    assert L.ecsim_cell_segments_static(None, 128, 128, 129, 1.0, 1.0, 1.0, 10, one, one, one, one, one) == -1
    text = L.ecsim_last_error().decode()
    assert "ECSIM_STATIC_MAX_CELLS" in text and str(limit) in text and "128 x 128 x 129" in text
    # the other argument checks
    assert L.ecsim_cell_segments_static(None, 1, 8, 8, 1.0, 1.0, 1.0, 10, one, one, one, one, one) == -1     # dims >= 2
    assert L.ecsim_cell_segments_static(None, 8, 8, 8, 0.0, 1.0, 1.0, 10, one, one, one, one, one) == -1     # spacing > 0
    assert L.ecsim_cell_segments_static(None, 8, 8, 8, 1.0, 1.0, 1.0, -1, one, one, one, one, one) == -1     # n >= 0
    assert L.ecsim_cell_segments_static(None, 8, 8, 8, 1.0, 1.0, 1.0, 10, None, one, one, one, one) == -1    # inputs
    assert L.ecsim_cell_segments_static(None, 8, 8, 8, 1.0, 1.0, 1.0, 10, one, one, one, None, None) == -1   # an output
