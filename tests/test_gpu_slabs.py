"""-m gpu: per-sub-domain execution of the interaction pass (PAPER.md L192,
L218-220, L226-228).  Every slab computes the rates of its own particles from its own range and its
two halo BUFFERS only (local cell table rebuilt from positions); over all slabs that must reproduce
the global pass value for value - the device-side proof that a halo one cell plane (2h) wide is
sufficient, and the first consumer of what a5 builds."""
import numpy as np
import pytest

from oracle import structure as OA
from paper_1210_1017_b200 import binding as B
from paper_1210_1017_b200 import workloads as W

from gpu_util import make_sph, oracle_rates, rate_errors

pytestmark = pytest.mark.gpu


def _global_then_slabs(w, n_slabs, planes=None):
    nc = OA.grid_dims(w.params["dom_min"], w.params["dom_max"], w.params["h"])
    planes = planes or W.slab_planes(nc[0], n_slabs)
    sph = make_sph(w)
    sph.sph_set_slabs(planes)
    sph.sph_sort_and_cells()
    sph.sph_build_halos()
    sph.sph_interact()
    ref = sph.sph_download(pos=False, vel=False, rho=False)
    T = sph.view_tensors()
    T["acc4"].fill_(float("nan"))                      # every entry must be rewritten by the slabs
    for s in range(len(planes) - 1):
        sph.sph_interact_slab(s)
    out = sph.sph_download(pos=False, vel=False, rho=False)
    assert sph.sph_status() == 0
    return ref, out


@pytest.mark.parametrize("nb,n_slabs", [(24, 3), (16, 2), (20, 5)])
def test_slabs_reproduce_the_global_pass_dam_break(nb, n_slabs):
    w = W.dam_break(nb, scrambled=True, n_slabs=n_slabs)
    ref, out = _global_then_slabs(w, n_slabs)
    assert np.array_equal(ref["acc"], out["acc"]) and np.array_equal(ref["drho"], out["drho"])
    # and the global pass itself is the oracle's (so the equality is not between two wrong results)
    ref_a, ref_d = oracle_rates(w)
    e_d, e_a = rate_errors(w, out["acc"], out["drho"], ref_a, ref_d)
    assert e_d <= 1e-4 and e_a <= 1e-4


def test_slabs_reproduce_the_global_pass_uniform_cube_8_slabs():
    w = W.uniform_cube(100003)
    ref, out = _global_then_slabs(w, 8)
    assert np.isfinite(out["drho"]).all()
    assert np.array_equal(ref["acc"], out["acc"]) and np.array_equal(ref["drho"], out["drho"])


def test_uneven_planes_and_single_slab():
    w = W.dam_break(16, scrambled=True, n_slabs=3)
    nc = OA.grid_dims(w.params["dom_min"], w.params["dom_max"], w.params["h"])
    planes = [0, 2, nc[0] - 2, nc[0]]                  # two minimal slabs at the ends
    ref, out = _global_then_slabs(w, 3, planes)
    assert np.array_equal(ref["acc"], out["acc"]) and np.array_equal(ref["drho"], out["drho"])
    ref, out = _global_then_slabs(w, 1)
    assert np.array_equal(ref["acc"], out["acc"]) and np.array_equal(ref["drho"], out["drho"])


@pytest.mark.parametrize("case", ["dense", "disordered"])
def test_slabs_vs_global_on_dense_and_disordered_states(case):
    """States whose tiles can overflow one candidate batch of the production kernel (IM_BATCH = 2176 for a
    nominal 2160): h = 3 dp (216 particles per cell, several batches per tile) and a disordered dam break.
    A tile that straddles a slab plane is then cut into batches at different candidates in the global and in
    the per-slab run (the global concatenation holds one x-row more), so the partial sums are added in a
    different order: equality is to rounding, not bit for bit.  Both must still be the oracle's rates."""
    if case == "dense":
        w = W.dam_break(14, scrambled=True)
        P = dict(w.params)
        P["h"] = W.f32(3.0 * P["dp"])
        lo = -2.0 * P["dp"] - 2.0 * P["h"]
        P["dom_min"] = (W.f32(lo),) * 3
        P["dom_max"] = tuple(W.f32(x + 2 * P["h"]) for x in w.params["dom_max"])
        w.params = P
        n_slabs = 2
    else:
        w = W.dam_break(32, scrambled=True)
        nf = w.n_fluid
        ids = np.arange(nf, dtype=np.int64)
        pos = w.pos.astype(np.float64)
        for c in range(3):
            pos[:nf, c] += (2.0 * W.u01(W.SEED_STATE + 7, ids, c) - 1.0) * 0.3 * w.params["dp"]
        w.pos = pos.astype(np.float32)
        n_slabs = 4
    ref, out = _global_then_slabs(w, n_slabs)
    s_a, s_d = np.abs(ref["acc"]).max(), np.abs(ref["drho"]).max()
    d_a, d_d = np.abs(ref["acc"] - out["acc"]).max() / s_a, np.abs(ref["drho"] - out["drho"]).max() / s_d
    same = np.array_equal(ref["acc"], out["acc"]) and np.array_equal(ref["drho"], out["drho"])
    print(f"slab vs global, {case}: bitwise {same}, max diff / max value: acc {d_a:.2e}, drho {d_d:.2e}")
    assert d_a <= 1e-5 and d_d <= 1e-5
    ref_a, ref_d = oracle_rates(w)
    e_d, e_a = rate_errors(w, out["acc"], out["drho"], ref_a, ref_d)
    assert e_d <= 1e-4 and e_a <= 1e-4


def test_slab_pass_needs_halos():
    w = W.dam_break(8, scrambled=True, n_slabs=2)
    sph = make_sph(w)
    sph.sph_sort_and_cells()
    with pytest.raises(B.SphError):
        sph.sph_interact_slab(0)
