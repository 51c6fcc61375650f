"""-m gpu test of sph_cell_table_static, the one entry point meant for callers that cannot allocate
device memory: code that is only lent the device pointers of a running simulation (an sph_view) and has
no workspace of its own, or that lives in a process where all GPU memory already belongs to someone
else's pool.  Its scratch is a fixed array inside the library, shared by every call on a GPU, so what
needs checking is (1) that it produces the very table the workspace-based path (sph_sort_and_cells)
produces, (2) that a call is not disturbed by what the previous call left in the shared array - hence
several calls in a row on different inputs, and (3) that it refuses sizes beyond the array instead of
overrunning it.

This file is named so that pytest collects it last: `pytest -x` stops at the first failure, and a failure
here must not hide the parity tests.  It has to pass on its own in a fresh process too (the first call on
a GPU is the one that looks up the array's device address), so nothing here relies on another test having
run before."""
import numpy as np
import pytest

from paper_1210_1017_b200 import workloads as W

from gpu_util import make_sph, u32

pytestmark = pytest.mark.gpu


def _sorted_state(w):
    """Existing path: sort + cell table out of a caller-allocated workspace.  Returns (sph, keyword tensor,
    ncells, reference cell table as numpy uint32)."""
    sph = make_sph(w, with_prev=False)
    sph.sph_sort_and_cells()
    T = sph.view_tensors()
    assert sph.sph_status() == 0
    return sph, T["keyword"], int(T["view"].ncells), u32(T["cell_begin"]).copy()


def _static_table(B, keyword, ncells):
    import torch
    # the caller's output buffer (inputs and outputs stay the caller's business); pre-filled so that an
    # entry the call failed to write shows up
    out = torch.full((ncells + 1,), -1, dtype=torch.int32, device=keyword.device)
    B.sph_cell_table_static(keyword, ncells, out)
    torch.cuda.synchronize()
    return u32(out)


def test_static_cell_table_equals_workspace_path_on_consecutive_calls():
    from paper_1210_1017_b200 import binding as B

    # A: a dam break inside a grid far larger than the tank, so the table has every kind of gap: short
    # ones filled inline, runs of > 32 empty cells (work list) and runs of > 65536 (several list entries)
    wa = W.dam_break(16)
    wa.params = dict(wa.params)
    lo, hi = wa.params["dom_min"], wa.params["dom_max"]
    wa.params["dom_max"] = (lo[0] + 2.0 * (hi[0] - lo[0]), lo[1] + 20.0 * (hi[1] - lo[1]), lo[2] + 20.0 * (hi[2] - lo[2]))
    sa, kw_a, nca, ref_a = _sorted_state(wa)
    assert 1 << 17 < nca <= B.SPH_STATIC_MAX_CELLS
    gaps = np.diff(np.flatnonzero(np.diff(ref_a.astype(np.int64)) > 0))
    assert gaps.max() > 32 and nca - (int(u32(kw_a)[-1]) & 0x0FFFFFFF) > 1 << 16

    # B: random positions filling their grid - a different table, few long gaps
    wb = W.uniform_cube(100003)
    sb, kw_b, ncb, ref_b = _sorted_state(wb)
    assert ncb <= B.SPH_STATIC_MAX_CELLS

    # calls in a row, all through the one shared array: A, B, A again, B again
    for kw, nc, ref in ((kw_a, nca, ref_a), (kw_b, ncb, ref_b), (kw_a, nca, ref_a), (kw_b, ncb, ref_b)):
        got = _static_table(B, kw, nc)
        assert got[-1] == kw.numel()
        assert np.array_equal(got, ref), "static-scratch cell table differs from the workspace path's"


def test_static_cell_table_limits_and_empty_input():
    import torch
    from paper_1210_1017_b200 import binding as B

    dev = torch.device("cuda:0")
    kw = torch.zeros(4, dtype=torch.int32, device=dev)
    too_many = B.SPH_STATIC_MAX_CELLS + 1
    out = torch.zeros(too_many + 1, dtype=torch.int32, device=dev)
    with pytest.raises(B.SphError) as ei:
        B.sph_cell_table_static(kw, too_many, out)
    assert ei.value.code == B.SPH_ERR_STATIC_LIMIT and "fixed scratch" in str(ei.value)
    torch.cuda.synchronize()
    assert int(out.abs().max().item()) == 0          # refused before anything was launched

    # the largest grid it accepts: 4 particles in cell 0, the other 2^22 - 1 cells empty (64 list entries)
    out = torch.full((B.SPH_STATIC_MAX_CELLS + 1,), -1, dtype=torch.int32, device=dev)
    B.sph_cell_table_static(kw, B.SPH_STATIC_MAX_CELLS, out)
    torch.cuda.synchronize()
    assert int(out[0].item()) == 0 and bool((out[1:] == 4).all().item())

    # no particles: an all-zero table
    out = torch.full((1001,), -1, dtype=torch.int32, device=dev)
    B.sph_cell_table_static(torch.empty(0, dtype=torch.int32, device=dev), 1000, out)
    torch.cuda.synchronize()
    assert int(out.abs().max().item()) == 0
