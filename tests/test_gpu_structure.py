"""-m gpu parity tests, structure part (a1-a6): the CUDA path through the C ABI against
ORACLE A, bit for bit, on seeded generator inputs."""
import numpy as np
import pytest

from oracle import structure as OA
from paper_1210_1017_b200 import workloads as W

from gpu_util import compare_structure, make_sph, u32

pytestmark = pytest.mark.gpu


def _planes(w, S=None):
    nc = OA.grid_dims(w.params["dom_min"], w.params["dom_max"], w.params["h"])
    return W.slab_planes(nc[0], S or w.n_slabs)


def test_config0_sort_cells_single_slab():
    w = W.dam_break(16)
    sph = make_sph(w)
    sph.sph_sort_and_cells()
    sph.sph_build_halos()
    A = compare_structure(sph, w, _planes(w, 1), None)
    assert len(A["migrants"]) == 0


@pytest.mark.parametrize("n", [1 << 16, 100003, 8191, 8192, 8193, 4095, 4097, 255, 256, 257, 1, 37])
def test_uniform_cube_sort_halos_migrants(n):
    """Random keys, 8 slabs, synthetic previous owners: several radix tiles and ragged tails
    (8192 = one radix tile exactly, 4096 = one migrant group, 256 = one gather tile, each also +-1)."""
    w = W.uniform_cube(n)
    nc = OA.grid_dims(w.params["dom_min"], w.params["dom_max"], w.params["h"])
    S = 8 if nc[0] >= 16 else 1
    planes = W.slab_planes(nc[0], S)
    if S == 1:
        w.prev_slab = np.zeros(n, dtype=np.uint8)
    sph = make_sph(w)
    sph.sph_set_slabs(planes)
    sph.sph_sort_and_cells()
    sph.sph_build_halos()
    A = compare_structure(sph, w, planes, w.prev_slab)
    if n >= 1 << 16:
        assert len(A["migrants"]) > 0 and all(len(L) + len(R) > 0 for L, R in A["halo"])


def test_second_sort_is_history_free_and_uses_previous_ranges():
    """A sort that starts from cell order (not id order) must give the same (cell, id) order;
    previous owners now come from the previous slab ranges: nothing moved => no migrants."""
    w = W.uniform_cube(50000)
    planes = _planes(w, 8)
    sph = make_sph(w)
    sph.sph_set_slabs(planes)
    sph.sph_sort_and_cells()
    sph.sph_sort_and_cells()
    sph.sph_build_halos()
    nc = OA.grid_dims(w.params["dom_min"], w.params["dom_max"], w.params["h"])
    cx, _, _ = OA.cell_coords(w.pos, w.params["dom_min"], w.params["h"], nc)
    own = OA.slab_of(cx, planes).astype(np.uint8)
    A = compare_structure(sph, w, planes, own)
    assert len(A["migrants"]) == 0


def test_dam_break_three_slabs_and_replaning():
    """Lattice block (many particles exactly on cell faces; jitter 1e-3 dp), boundary particles,
    3 slabs; then new planes through sph_build_halos only (edge labels recomputed, no re-sort)."""
    w = W.dam_break(24, n_slabs=3)
    planes = _planes(w, 3)
    sph = make_sph(w)
    sph.sph_build_halos  # noqa: B018  (needs a sort first, checked below)
    from paper_1210_1017_b200.binding import SphError
    with pytest.raises(SphError):
        sph.sph_build_halos(planes)
    with pytest.raises(SphError):
        sph.sph_interact()
    sph.sph_set_slabs(planes)
    sph.sph_sort_and_cells()
    sph.sph_build_halos()
    compare_structure(sph, w, planes, None)
    planes2 = [0, 4, planes[-1] - 5, planes[-1]]
    sph.sph_build_halos(planes2)
    compare_structure(sph, w, planes2, None)
    for bad in ([0, 1, planes[-1]], [0, 5, 5, planes[-1]], [1, 5, planes[-1]], [0, 5, planes[-1] + 1]):
        with pytest.raises(SphError):
            sph.sph_build_halos(bad)


def test_degenerate_inputs():
    # all particles in one cell, some outside the grid (clamped, never dropped)
    w = W.uniform_cube(5000)
    w.pos[:] = w.pos * np.float32(1e-4) + np.float32(0.5)
    w.pos[:7] = [[-3.0, 0.5, 0.5], [9.0, 9.0, 9.0], [0.5, -1.0, 2.0], [1.0, 1.0, 1.0],
                 [0.0, 0.0, 0.0], [-0.0, 0.999999, 1e-30], [0.25, 0.25, -1e-30]]
    w.prev_slab = None
    planes = _planes(w, 4)
    sph = make_sph(w)
    sph.sph_set_slabs(planes)
    sph.sph_sort_and_cells()
    sph.sph_build_halos()
    compare_structure(sph, w, planes, None)
    # non-finite positions raise the sticky device flag
    w.pos[3, 1] = np.nan
    sph.sph_set_state(w.pos, w.vel, w.rho, w.type)
    assert sph.sph_status() == -6


def test_four_radix_passes_sparse_grid():
    """> 2^24 cells (4 digit passes) with few particles: long runs of empty cells in the table."""
    w = W.uniform_cube(20000)
    P = dict(w.params)
    P["h"] = W.f32(0.5 / 260.0)          # 260^3 = 17.6 M cells -> 25 key bits
    P["dp"] = P["h"]
    w.params = P
    nc = OA.grid_dims(P["dom_min"], P["dom_max"], P["h"])
    assert nc[0] * nc[1] * nc[2] > (1 << 24)
    planes = W.slab_planes(nc[0], 16)
    sph = make_sph(w)
    assert sph.sph_get_view().cell_bits == 25
    sph.sph_set_slabs(planes)
    sph.sph_sort_and_cells()
    sph.sph_build_halos()
    compare_structure(sph, w, planes, w.prev_slab // 1)   # prev owners in 0..7 of 16 slabs


def test_config1_full_size_structure():
    """BASELINE config 1 (1.2 M particles, 3 slabs) at full size, complete comparison."""
    w = W.dam_break(100)
    planes = _planes(w)
    sph = make_sph(w)
    sph.sph_set_slabs(planes)
    sph.sph_sort_and_cells()
    sph.sph_build_halos()
    compare_structure(sph, w, planes, None)


def test_micro_16m_structure_properties_and_samples():
    """Sort/halo microbenchmark size 2^24: full oracle order (numpy lexsort) compared on the
    whole permutation; cell table via searchsorted."""
    w = W.uniform_cube(1 << 24)
    planes = _planes(w, 8)
    sph = make_sph(w)
    sph.sph_set_slabs(planes)
    sph.sph_sort_and_cells()
    sph.sph_build_halos()
    compare_structure(sph, w, planes, w.prev_slab, check_payload=False)


def test_micro_64m_full_structure():
    """Sort/halo microbenchmark size 2^26 (3 radix passes at full tile counts): the complete structure
    comparison (numpy lexsort of 67 M keys)."""
    w = W.uniform_cube(1 << 26)
    planes = _planes(w, 8)
    sph = make_sph(w)
    sph.sph_set_slabs(planes)
    sph.sph_sort_and_cells()
    sph.sph_build_halos()
    compare_structure(sph, w, planes, w.prev_slab, check_payload=False)


def test_micro_256m_four_pass_sort_by_its_defining_properties():
    """2^28 particles, 26 key bits = 4 radix passes at full tile counts.  Instead of a 268 M-element
    lexsort the result is checked through the three properties that define it uniquely: (i) the ids are
    a permutation, (ii) every sorted keyword is ORACLE A's keyword of that id, (iii) the sequence is
    strictly increasing in (cell, id).  The cell table is checked against searchsorted on the (then
    proven) sorted cells, the slab ranges against it."""
    n = 1 << 28
    w = W.uniform_cube(n)
    P = w.params
    planes = _planes(w, 8)
    sph = make_sph(w)
    v = sph.sph_get_view()
    assert v.cell_bits == 26
    sph.sph_set_slabs(planes)
    sph.sph_sort_and_cells()
    sph.sph_build_halos()
    assert sph.sph_status() == 0
    T = sph.view_tensors()
    kw = u32(T["keyword"])
    ids = (u32(T["idt"]) & 0x0FFFFFFF).astype(np.int64)
    assert np.array_equal(np.bincount(ids, minlength=n), np.ones(n, dtype=np.int64))            # (i)
    nc = OA.grid_dims(P["dom_min"], P["dom_max"], P["h"])
    kw_by_id, cell_by_id = OA.keywords(w.pos, P["dom_min"], P["h"], nc, planes, w.prev_slab)
    assert np.array_equal(kw, kw_by_id[ids])                                                    # (ii)
    cell = (kw & 0x0FFFFFFF).astype(np.int64)
    comp = cell * n + ids                                                                       # < 2^54
    assert (np.diff(comp) > 0).all()                                                            # (iii)
    del comp, kw_by_id, cell_by_id
    ncells = nc[0] * nc[1] * nc[2]
    begin, _ = OA.cell_table(cell, ncells)
    assert np.array_equal(u32(T["cell_begin"]), begin)
    assert np.array_equal(u32(T["slab_begin"]), begin[np.asarray(planes, dtype=np.int64) * nc[1] * nc[2]])
    # migrants: count and records against the linear filter over the sorted sequence
    slab_s = OA.slab_of(cell // (nc[1] * nc[2]), planes)
    prev_s = w.prev_slab[ids].astype(np.int64)
    m = np.nonzero(prev_s != slab_s)[0]
    mig = u32(T["migrants"]).astype(np.int64).reshape(-1, 4)
    assert len(mig) == len(m) > 0
    assert np.array_equal(mig, np.stack([ids[m], m, prev_s[m], slab_s[m]], axis=1))
