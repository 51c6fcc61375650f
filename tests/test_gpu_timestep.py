"""-m gpu parity tests of the variable time step (NEXT-1 of SURVEY 8(f); PAPER.md L150, L222;
DESIGN.md reading A8b): the CUDA reduction through the C ABI against ORACLE B.

max_j |mu_ij| is discontinuous in the cut-off radius (|mu| does not vanish at r = 2h, and a
lattice has many pairs exactly there), so the fp32 result is bracketed between the oracle's values
for cut = 1 -+ 1e-5 instead of being compared with one number (several results are valid; what
must hold is that every pair clearly inside counts and no pair clearly outside does)."""
import numpy as np
import pytest

from oracle import physics as OB
from oracle import structure as OA
from paper_1210_1017_b200 import binding as B
from paper_1210_1017_b200 import workloads as W

from gpu_util import make_sph, rel_l2

pytestmark = pytest.mark.gpu
CFL = 0.2
EPS = 1e-5


def _slab_of(w, planes):
    P = w.params
    A = OA.structure(w.pos, np.arange(w.n), P["dom_min"], P["dom_max"], P["h"], planes)
    cell_sorted = A["keyword_sorted"] & 0x0FFFFFFF
    nc = A["nc"]
    cx = cell_sorted // (nc[1] * nc[2])
    slab_sorted = np.searchsorted(np.asarray(planes), cx, side="right") - 1
    slab = np.empty(w.n, dtype=np.int64)
    slab[A["id_sorted"]] = slab_sorted
    return slab


def test_some_case_has_a_ragged_last_warp():
    assert any(W.dam_break(nb).n % 32 != 0 for nb in (16, 13))


@pytest.mark.parametrize("variant", [0, 1])
@pytest.mark.parametrize("n_slabs,nb", [(1, 16), (3, 16), (3, 13)])
def test_time_step_matches_oracle_bracket(variant, n_slabs, nb):
    w = W.dam_break(nb, scrambled=True, n_slabs=n_slabs)
    nc = OA.grid_dims(w.params["dom_min"], w.params["dom_max"], w.params["h"])
    planes = W.slab_planes(nc[0], n_slabs)
    sph = make_sph(w)
    sph.sph_set_option(B.SPH_OPT_INTERACT_VARIANT, variant)
    sph.sph_set_option(B.SPH_OPT_ADAPTIVE_DT, 1)
    sph.sph_set_slabs(planes)
    sph.sph_sort_and_cells()
    sph.sph_interact()
    dt, amax, smax = sph.sph_time_step(CFL)
    assert sph.sph_status() == 0
    p = OB.params_from_workload(w.params)
    acc, _ = OB.rates(p, w.pos, w.vel, w.rho, w.type)
    slab = _slab_of(w, planes)
    lo = OB.time_step(p, w.pos, w.vel, w.rho, w.type, acc, CFL, cut=1.0 - EPS, slab_of=slab, n_slabs=n_slabs)
    hi = OB.time_step(p, w.pos, w.vel, w.rho, w.type, acc, CFL, cut=1.0 + EPS, slab_of=slab, n_slabs=n_slabs)
    assert len(amax) == n_slabs
    assert np.all(np.abs(amax - lo["amax_slab"]) <= 1e-4 * lo["amax_slab"].max())
    assert np.all(smax >= lo["smax_slab"] * (1 - 1e-5)) and np.all(smax <= hi["smax_slab"] * (1 + 1e-5))
    assert hi["dt"] * (1 - 1e-4) <= dt <= lo["dt"] * (1 + 1e-4)
    # the viscous signal really contributes in this state (else the check is vacuous)
    c_max = OB.sound_speed(p, float(w.rho.max()))
    assert lo["smax_slab"].max() > 1.02 * c_max


@pytest.mark.parametrize("variant", [0, 1])
def test_mumax_per_particle_on_a_disordered_state(variant):
    """The filter of the production kernel must never drop a pair with r < 2h (reading A19): a
    lost pair just inside the cut-off changes a rate by ~1e-6 of a term - invisible at 1e-4 - but it can be
    the pair that sets max_j |mu_ij| (L112, L150), which does not vanish at r = 2h.  So mumax is compared
    PARTICLE BY PARTICLE with the oracle's bracket: at least the maximum over the pairs clearly inside
    (cut = 1 - 1e-5), at most the one over the pairs up to just outside (cut = 1 + 1e-5)."""
    w = W.dam_break(32, scrambled=True)
    nf = w.n_fluid
    ids = np.arange(nf, dtype=np.int64)
    pos = w.pos.astype(np.float64)
    for c in range(3):
        pos[:nf, c] += (2.0 * W.u01(W.SEED_STATE + 7, ids, c) - 1.0) * 0.3 * w.params["dp"]
    w.pos = pos.astype(np.float32)
    sph = make_sph(w)
    sph.sph_set_option(B.SPH_OPT_INTERACT_VARIANT, variant)
    sph.sph_set_option(B.SPH_OPT_ADAPTIVE_DT, 1)
    sph.sph_sort_and_cells()
    sph.sph_interact()
    T = sph.view_tensors()
    assert sph.sph_status() == 0
    order = T["idt"].cpu().numpy().view(np.uint32) & 0x0FFFFFFF
    mu = np.empty(w.n, dtype=np.float64)
    mu[order] = T["mumax"].cpu().numpy()
    p = OB.params_from_workload(w.params)
    acc, _ = OB.rates(p, w.pos, w.vel, w.rho, w.type)
    lo = OB.time_step(p, w.pos, w.vel, w.rho, w.type, acc, CFL, cut=1.0 - EPS)["mu"]
    hi = OB.time_step(p, w.pos, w.vel, w.rho, w.type, acc, CFL, cut=1.0 + EPS)["mu"]
    scale = hi.max()
    assert scale > 0 and (lo > 0).mean() > 0.5
    tol = 2e-5 * scale                               # fp32 evaluation of h v.r / (r^2 + eta^2)
    worst_lo, worst_hi = (lo - mu).max() / scale, (mu - hi).max() / scale
    print(f"mumax per particle, variant {variant}: below lower bracket by {worst_lo:.2e}, above upper by {worst_hi:.2e} (of max mu)")
    assert np.all(mu >= lo - tol), "a pair inside the cut-off was lost"
    assert np.all(mu <= hi + tol), "a pair outside the cut-off was counted"


def test_time_step_needs_mu():
    w = W.dam_break(8, scrambled=True)
    sph = make_sph(w)
    sph.sph_sort_and_cells()
    sph.sph_interact()                       # fixed-dt path: no mu recorded
    with pytest.raises(B.SphError):
        sph.sph_time_step(CFL)


def test_adaptive_steps_follow_the_oracle():
    """Ten adaptive steps: the oracle steps with ITS OWN dt each step; dt sequences and states agree."""
    w = W.dam_break(12, scrambled=True, n_slabs=2)
    w.params = dict(w.params)
    w.params["verlet_ns"] = 4
    nc = OA.grid_dims(w.params["dom_min"], w.params["dom_max"], w.params["h"])
    sph = make_sph(w)
    sph.sph_set_slabs(W.slab_planes(nc[0], 2))
    p = OB.params_from_workload(w.params)
    s = OB.State(w.pos, w.vel, w.rho, w.type)
    for k in range(10):
        dt_gpu = sph.sph_step_adaptive(CFL)
        acc, _ = OB.rates(p, s.r, s.v, s.rho, s.type)
        o = OB.time_step(p, s.r, s.v, s.rho, s.type, acc, CFL)
        assert abs(dt_gpu - o["dt"]) <= 1e-3 * o["dt"], (k, dt_gpu, o["dt"])
        OB.step(p, s, o["dt"], verlet_ns=w.params["verlet_ns"])
    out = sph.sph_download()
    assert sph.sph_status() == 0
    fl = w.type == 0
    assert rel_l2(out["pos"], s.r) <= 1e-3
    assert rel_l2(out["rho"], s.rho) <= 1e-3
    assert rel_l2(out["vel"][fl], s.v[fl]) <= 1e-3
