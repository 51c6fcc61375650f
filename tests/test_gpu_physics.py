"""-m gpu parity tests, physics part (a7-a8): fp32 CUDA path through the C ABI against the fp64
ORACLE B on the same seeded inputs.

Tolerances (BASELINE.json north_star): one step - max|err| / max|value| <= 1e-4 separately for
d rho/dt (all particles) and acceleration (fluid); ten steps - relative L2 <= 1e-3 for r, v, rho
(plus the displacement r - r0, which ||r|| would hide)."""
import numpy as np
import pytest

from oracle import physics as OB
from oracle import structure as OA
from paper_1210_1017_b200 import workloads as W

from gpu_util import make_sph, oracle_rates, rate_errors, rel_l2

pytestmark = pytest.mark.gpu

TOL_RATE = 1e-4
TOL_STATE = 1e-3


def _gpu_rates(w, variant=0, planes=None):
    sph = make_sph(w)
    sph.sph_set_option(0, variant)
    if planes is not None:
        sph.sph_set_slabs(planes)
    sph.sph_sort_and_cells()
    sph.sph_interact()
    out = sph.sph_download()
    assert sph.sph_status() == 0
    return out


@pytest.mark.parametrize("variant", [0, 1])
def test_config0_rest_state_rates(variant):
    """Prescribed check: config 0 at rest.  p = 0 and v = 0, so every fluid rate is (g, 0)."""
    w = W.dam_break(16)
    ref_a, ref_d = oracle_rates(w)
    out = _gpu_rates(w, variant)
    e_d, e_a = rate_errors(w, out["acc"], out["drho"], ref_a, ref_d)
    assert e_d <= TOL_RATE and e_a <= TOL_RATE
    assert (out["acc"][w.type == 1] == 0).all()
    # download returns the inputs unchanged in id order
    assert np.array_equal(out["pos"], w.pos) and np.array_equal(out["rho"], w.rho)


@pytest.mark.parametrize("variant", [0, 1])
def test_disordered_positions_rates(variant):
    """No lattice: every fluid particle is moved by U(-0.3, 0.3) dp per axis (seeded), on top of random
    velocities and densities.  Neighbour counts then differ from particle to particle (the lanes of a warp
    drain different numbers of pairs), pairs sit anywhere around the cut-off instead of exactly at 2h, and
    cells hold 20-35 particles instead of 27."""
    w = W.dam_break(32, scrambled=True)
    nf = w.n_fluid
    ids = np.arange(nf, dtype=np.int64)
    dp = w.params["dp"]
    pos = w.pos.astype(np.float64)
    for c in range(3):
        pos[:nf, c] += (2.0 * W.u01(W.SEED_STATE + 7, ids, c) - 1.0) * 0.3 * dp
    w.pos = pos.astype(np.float32)
    ref_a, ref_d = oracle_rates(w)
    out = _gpu_rates(w, variant)
    e_d, e_a = rate_errors(w, out["acc"], out["drho"], ref_a, ref_d)
    assert e_d <= TOL_RATE, e_d
    assert e_a <= TOL_RATE, e_a


@pytest.mark.parametrize("variant", [0, 1])
@pytest.mark.parametrize("nb", [16, 40])
def test_scrambled_state_rates(variant, nb):
    """Reading A21: same positions, random velocities and densities, so that pressure,
    viscosity (both branches) and continuity are all exercised.  nb = 40 spans many CTAs."""
    w = W.dam_break(nb, scrambled=True)
    ref_a, ref_d = oracle_rates(w)
    assert np.abs(ref_d).max() > 0 and np.abs(ref_a[w.type == 0]).max() > 10
    out = _gpu_rates(w, variant)
    e_d, e_a = rate_errors(w, out["acc"], out["drho"], ref_a, ref_d)
    assert e_d <= TOL_RATE, e_d
    assert e_a <= TOL_RATE, e_a


def test_variants_agree_and_slabs_do_not_change_rates():
    w = W.dam_break(24, scrambled=True, n_slabs=3)
    nc = OA.grid_dims(w.params["dom_min"], w.params["dom_max"], w.params["h"])
    a = _gpu_rates(w, 0)
    b = _gpu_rates(w, 1)
    c = _gpu_rates(w, 0, planes=W.slab_planes(nc[0], 3))
    s = np.abs(b["acc"]).max()
    assert np.abs(a["acc"] - b["acc"]).max() <= 2e-5 * s
    assert np.abs(a["drho"] - b["drho"]).max() <= 2e-5 * np.abs(b["drho"]).max()
    assert np.array_equal(a["acc"], c["acc"]) and np.array_equal(a["drho"], c["drho"])


@pytest.mark.parametrize("variant", [0, 1])
def test_nonuniform_mass_and_cubic_spline(variant):
    w = W.dam_break(12, scrambled=True)
    w.params = dict(w.params)
    w.params["mass_bound"] = W.f32(0.6 * w.params["mass_fluid"])
    ref_a, ref_d = oracle_rates(w)
    out = _gpu_rates(w, variant)
    e_d, e_a = rate_errors(w, out["acc"], out["drho"], ref_a, ref_d)
    assert e_d <= TOL_RATE and e_a <= TOL_RATE
    w.params["kernel"] = 1                       # the paper's own kernel (L81)
    ref_a, ref_d = oracle_rates(w)
    out = _gpu_rates(w, variant)
    e_d, e_a = rate_errors(w, out["acc"], out["drho"], ref_a, ref_d)
    assert e_d <= TOL_RATE and e_a <= TOL_RATE


def test_dense_cells_use_several_batches_and_chunks():
    """Cells far denser than the kernel is tuned for (h = 3 dp: 216 per cell): more targets
    than threads per z-block and more candidates than one staging batch."""
    w = W.dam_break(14, scrambled=True)
    P = dict(w.params)
    P["h"] = W.f32(3.0 * P["dp"])
    lo = -2.0 * P["dp"] - 2.0 * P["h"]
    P["dom_min"] = (W.f32(lo),) * 3
    P["dom_max"] = tuple(W.f32(x + 2 * P["h"]) for x in w.params["dom_max"])
    w.params = P
    ref_a, ref_d = oracle_rates(w)
    out = _gpu_rates(w, 0)
    e_d, e_a = rate_errors(w, out["acc"], out["drho"], ref_a, ref_d)
    assert e_d <= TOL_RATE and e_a <= TOL_RATE


def test_particles_outside_the_grid_switch_the_filter_to_wide():
    """Reading A13: particles beyond the grid sit clamped in edge cells.  The production kernel's tf32
    distance filter (interact_mma.cu, filter_thr) is derived for records inside the staged region of their
    tile (|x|, |y| <= 4h, |z| <= (zb + 2) h from the tile centre); a tile that meets a record outside that
    model sets its "wide" switch (ImStage::wide), which lets every candidate through to the exact fp32 pair
    term.  Here the grid stops at a third of the tank in x, so the far wall and part of the floor are up to
    ~17 h outside: the limit reached is the wide switch of the production kernel."""
    w = W.dam_break(12, scrambled=True)
    P = dict(w.params)
    P["dom_max"] = (W.f32(P["dom_min"][0] + 10.0 * 2.0 * P["h"]), P["dom_max"][1], P["dom_max"][2])
    w.params = P
    assert (w.pos[:, 0] > P["dom_max"][0] + 8.0 * P["h"]).any()
    ref_a, ref_d = oracle_rates(w)
    out = _gpu_rates(w, 0)
    e_d, e_a = rate_errors(w, out["acc"], out["drho"], ref_a, ref_d)
    assert e_d <= TOL_RATE and e_a <= TOL_RATE


def test_sparse_cells_long_z_blocks():
    """h = 0.75 dp: 3.4 particles per cell, so a tile of the production kernel takes its longest z-block
    (zb = IM_ZMAX = 6 cells: the tf32 error model at its widest, |z| <= 8 h, and its largest threshold pad);
    variant 1, the plain 27-cell walk, is the second opinion."""
    w = W.dam_break(16, scrambled=True)
    P = dict(w.params)
    P["h"] = W.f32(0.75 * P["dp"])
    w.params = P
    ref_a, ref_d = oracle_rates(w)
    assert np.abs(ref_d).max() > 0
    out = _gpu_rates(w, 0)
    e_d, e_a = rate_errors(w, out["acc"], out["drho"], ref_a, ref_d)
    assert e_d <= TOL_RATE and e_a <= TOL_RATE
    b = _gpu_rates(w, 1)
    assert np.abs(out["drho"] - b["drho"]).max() <= 2e-5 * np.abs(b["drho"]).max()


def _run_ten_steps(w, steps=10):
    sph = make_sph(w)
    nc = OA.grid_dims(w.params["dom_min"], w.params["dom_max"], w.params["h"])
    sph.sph_set_slabs(W.slab_planes(nc[0], w.n_slabs))
    p = OB.params_from_workload(w.params)
    s = OB.State(w.pos, w.vel, w.rho, w.type)
    for _ in range(steps):
        sph.sph_step(w.dt)
        OB.step(p, s, w.dt, verlet_ns=w.params["verlet_ns"])
    out = sph.sph_download()
    assert sph.sph_status() == 0
    return out, s


def test_config0_ten_steps():
    """Prescribed check: config 0, 10 Verlet steps from rest (corrective step 0 + 9 ordinary)."""
    w = W.dam_break(16)
    out, s = _run_ten_steps(w)
    assert rel_l2(out["pos"], s.r) <= TOL_STATE
    assert rel_l2(out["rho"], s.rho) <= TOL_STATE
    fl = w.type == 0
    assert rel_l2(out["vel"][fl], s.v[fl]) <= TOL_STATE
    disp_ref = s.r[fl] - w.pos[fl].astype(np.float64)
    disp = out["pos"][fl].astype(np.float64) - w.pos[fl].astype(np.float64)
    assert np.linalg.norm(disp - disp_ref) <= 5e-3 * np.linalg.norm(disp_ref)
    assert np.array_equal(out["pos"][~fl], w.pos[~fl])          # boundary particles never move


def test_scrambled_ten_steps_with_corrective_period_and_slabs():
    """Scrambled start, verlet_ns = 4 (both integrator branches several times), 3 slabs rebuilt
    every step; the last step's rates are compared too."""
    w = W.dam_break(16, scrambled=True, n_slabs=3)
    w.params = dict(w.params)
    w.params["verlet_ns"] = 4
    out, s = _run_ten_steps(w)
    fl = w.type == 0
    assert rel_l2(out["pos"], s.r) <= TOL_STATE
    assert rel_l2(out["rho"], s.rho) <= TOL_STATE
    assert rel_l2(out["vel"][fl], s.v[fl]) <= TOL_STATE
    disp_ref = s.r[fl] - w.pos[fl].astype(np.float64)
    disp = out["pos"][fl].astype(np.float64) - w.pos[fl].astype(np.float64)
    assert np.linalg.norm(disp - disp_ref) <= TOL_STATE * np.linalg.norm(disp_ref)
    # rates used by step 10 (acc4 still holds them): fp32 trajectory vs fp64 trajectory
    assert rel_l2(out["acc"][fl], s.acc[fl]) <= 5e-3
    assert rel_l2(out["drho"], s.drho) <= 5e-3


@pytest.mark.parametrize("kernel", [0, 1])
def test_config1_full_size_sampled_rates(kernel):
    """BASELINE config 1 (1.2 M particles) at full size, scrambled state, in the launch
    configuration bench.py uses; the oracle evaluates a sample of particles one neighbourhood
    at a time (all particles within 2h of the sample, brute force).  kernel = 1: the cubic spline the
    paper itself used (L81; NEXT-2 of SURVEY 8(f)) at the same size."""
    w = W.dam_break(100, scrambled=True)
    w.params = dict(w.params)
    w.params["kernel"] = kernel
    out = _gpu_rates(w, 0)
    p = OB.params_from_workload(w.params)
    rng_ids = (W.u01(77, np.arange(64), 0) * w.n).astype(np.int64)
    two_h = 2.0 * w.params["h"]
    pos64 = w.pos.astype(np.float64)
    worst_a, worst_d, scale_a, scale_d = 0.0, 0.0, 0.0, 0.0
    for i in rng_ids:
        near = np.nonzero((np.abs(pos64 - pos64[i]) <= two_h * 1.001).all(axis=1))[0]
        k = int(np.nonzero(near == i)[0][0])
        a, d = OB.rates(p, w.pos[near], w.vel[near], w.rho[near], w.type[near], mode=0)
        worst_a = max(worst_a, np.abs(out["acc"][i] - a[k]).max())
        worst_d = max(worst_d, abs(out["drho"][i] - d[k]))
        scale_a = max(scale_a, np.abs(a[k]).max())
        scale_d = max(scale_d, abs(d[k]))
    assert worst_a <= TOL_RATE * scale_a and worst_d <= TOL_RATE * scale_d


def test_moving_wall_particles_are_not_integrated_but_act_on_the_fluid():
    """boundary particles obey the same equations as the fluid, but "the integration update for
    position and velocity is not performed" (their motion is "externally imposed").  The wall particles of a
    dam break are given a velocity: after sph_step their r and v must keep their bits while their density
    moves; the fluid next to them must feel the wall's velocity (its d rho/dt differs from the static-wall
    value) and still match ORACLE B to the one-step tolerance."""
    w = W.dam_break(16, scrambled=True)
    bd = w.type == 1
    ids = np.arange(w.n, dtype=np.int64)
    w_static_d = oracle_rates(w)[1]
    for c in range(3):
        w.vel[bd, c] = ((2.0 * W.u01(W.SEED_STATE + 11, ids[bd], c) - 1.0) * 0.5).astype(np.float32)
    ref_a, ref_d = oracle_rates(w)
    fl = ~bd
    assert np.abs(ref_d[fl] - w_static_d[fl]).max() > 1e-2 * np.abs(ref_d).max()
    sph = make_sph(w)
    sph.sph_sort_and_cells()
    sph.sph_interact()
    out = sph.sph_download()
    e_d, e_a = rate_errors(w, out["acc"], out["drho"], ref_a, ref_d)
    assert e_d <= TOL_RATE and e_a <= TOL_RATE, (e_d, e_a)
    s = OB.State(w.pos, w.vel, w.rho, w.type)
    p = OB.params_from_workload(w.params)
    for _ in range(3):
        sph.sph_step(w.dt)
        OB.step(p, s, w.dt, verlet_ns=w.params["verlet_ns"])
    out = sph.sph_download(acc=False, drho=False)
    assert sph.sph_status() == 0
    assert np.array_equal(out["pos"][bd].view(np.uint32), w.pos[bd].view(np.uint32))      # bit-unchanged
    assert np.array_equal(out["vel"][bd].view(np.uint32), w.vel[bd].view(np.uint32))
    assert (out["rho"][bd] != w.rho[bd]).mean() > 0.5
    assert rel_l2(out["rho"][bd] - w.rho[bd].astype(np.float64), s.rho[bd] - w.rho[bd]) <= 1e-2
    assert rel_l2(out["rho"], s.rho) <= TOL_STATE and rel_l2(out["vel"][fl], s.v[fl]) <= TOL_STATE
