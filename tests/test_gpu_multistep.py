"""-m gpu: stage-wise multi-step structure parity with REAL migrants (SURVEY 8(c) "For multi-step runs the
check is stage-wise"; PAPER.md L198-210 the per-step "migrate" stage, L264 migration labels), re-planing
with migrants, and movable slab planes.

At every step k the CUDA path's OWN pre-sort fp32 positions (sph_download) and the owners of step k-1
are fed to ORACLE A; keywords, permutation, cell table, slab ranges, halo buffers (ids and copied bits),
migrant records and counts must agree bit for bit.  This is where the key kernel's "previous owner =
slab range of the last sort" branch (the one sph_step runs) meets the oracle with a non-empty answer."""
import dataclasses

import numpy as np
import pytest

from oracle import structure as OA
from paper_1210_1017_b200 import binding as B
from paper_1210_1017_b200 import workloads as W

from gpu_util import compare_structure, make_sph, owners_by_id, u32

pytestmark = pytest.mark.gpu


def _violent_dam_break(nb=20, n_slabs=5):
    """Scrambled dam break with velocities x20 and thin slabs over the fluid block: with 4 dt per step
    a few hundred particles cross slab planes every step (tuned with the oracle: densities stay > 0
    for 12 steps)."""
    w = W.dam_break(nb, scrambled=True, n_slabs=n_slabs)
    w.vel = (w.vel * np.float32(20.0)).astype(np.float32)
    nc = OA.grid_dims(w.params["dom_min"], w.params["dom_max"], w.params["h"])
    planes = [0] + [2 * k for k in range(1, n_slabs)] + [nc[0]]
    return w, nc, planes


def _state(sph):
    out = sph.sph_download(acc=False, drho=False)
    return out["pos"], out["vel"], out["rho"]


def test_stage_wise_structure_with_real_migrants_and_a_replane():
    w, nc, planes = _violent_dam_break()
    dt = 4.0 * w.dt
    sph = make_sph(w, with_prev=False)
    sph.sph_set_slabs(planes)
    prev = None
    total_mig = steps_with_mig = 0
    for k in range(6):
        pos, vel, rho = _state(sph)                      # the state the step's sort will see
        sph.sph_step(dt)
        wk = dataclasses.replace(w, pos=pos, vel=vel, rho=rho)
        A = compare_structure(sph, wk, planes, prev, check_payload=False, check_halo_payload=True)
        assert A["owned"].sum() == w.n
        total_mig += len(A["migrants"])
        steps_with_mig += len(A["migrants"]) > 0
        prev = owners_by_id(A, w.n)
    assert steps_with_mig >= 3 and total_mig > 300

    # step 6 by hand: sort, halos; then NEW planes without a new sort (owners change because planes
    # move: migrants across more than one slab, reading A15); then the rest of the step
    pos, vel, rho = _state(sph)
    wk = dataclasses.replace(w, pos=pos, vel=vel, rho=rho)
    sph.sph_sort_and_cells()
    sph.sph_build_halos()
    A = compare_structure(sph, wk, planes, prev)
    planes2 = [0, 3, 5, 9, 12, nc[0]]
    sph.sph_build_halos(planes2)
    A2 = compare_structure(sph, wk, planes2, prev)
    mig = A2["migrants"]
    assert len(mig) > len(A["migrants"]) and np.count_nonzero(np.abs(mig[:, 2] - mig[:, 3]) > 1) > 0
    # re-planing back and forth leaves no trace
    sph.sph_build_halos(planes)
    compare_structure(sph, wk, planes, prev)
    sph.sph_build_halos(planes2)
    compare_structure(sph, wk, planes2, prev)
    prev = owners_by_id(A2, w.n)
    # the step's own sort sees unmoved particles whose previous owners are the NEW planes' ranges
    sph.sph_step(dt)
    A = compare_structure(sph, wk, planes2, prev, check_payload=False, check_halo_payload=True)
    assert len(A["migrants"]) == 0
    for k in range(4):
        pos, vel, rho = _state(sph)
        sph.sph_step(dt)
        wk = dataclasses.replace(w, pos=pos, vel=vel, rho=rho)
        A = compare_structure(sph, wk, planes2, prev, check_payload=False, check_halo_payload=True)
        total_mig += len(A["migrants"])
        prev = owners_by_id(A, w.n)
    assert sph.sph_status() == 0


def test_first_sort_replane_has_no_migrants():
    """Reading A15: without previous owners nothing migrates, whatever planes are applied later."""
    w, nc, planes = _violent_dam_break(16, 3)
    sph = make_sph(w, with_prev=False)
    sph.sph_set_slabs(planes)
    sph.sph_sort_and_cells()
    sph.sph_build_halos([0, 5, 9, nc[0]])
    A = compare_structure(sph, w, [0, 5, 9, nc[0]], None)
    assert len(A["migrants"]) == 0


def test_balance_planes_match_the_oracle_and_equalise():
    """sph_balance_slabs == OA.balance_planes on the plane counts of the same positions; a dam break
    (fluid in the left third) gets narrower slabs on the left."""
    for nb, S in ((20, 4), (24, 3), (16, 8)):
        w = W.dam_break(nb, n_slabs=S)
        P = w.params
        nc = OA.grid_dims(P["dom_min"], P["dom_max"], P["h"])
        sph = make_sph(w, with_prev=False)
        with pytest.raises(B.SphError):
            sph.sph_balance_slabs(S)                      # needs a sort
        even = [int(x) for x in W.slab_planes(nc[0], S)]
        sph.sph_set_slabs(even)
        sph.sph_sort_and_cells()
        got = sph.sph_balance_slabs(S)
        exp = OA.balance_planes(OA.plane_counts(w.pos, P["dom_min"], P["dom_max"], P["h"]), S)
        assert got == exp
        if nc[0] >= 2 * S + 2:
            sph.sph_build_halos(got)
            A = compare_structure(sph, w, got, None)
            Aeven = OA.structure(w.pos, np.arange(w.n), P["dom_min"], P["dom_max"], P["h"], even)
            assert A["owned"].max() <= Aeven["owned"].max()
    with pytest.raises(B.SphError):
        sph.sph_balance_slabs(17)


def test_dam_break_rebalanced_every_20_steps():
    """200 steps of a small dam break, planes re-chosen every 20 steps from the cell table: at each
    re-balance the planes equal the oracle's bit for bit, sum(owned) = N, migrants (incl. moves across
    more than one slab when planes jump) match, and the per-slab interaction pass over the NEW slabs
    still equals the global pass."""
    w = W.dam_break(16, scrambled=True, n_slabs=4)
    w.vel = (w.vel * np.float32(10.0)).astype(np.float32)
    P = w.params
    nc = OA.grid_dims(P["dom_min"], P["dom_max"], P["h"])
    S = 4
    planes = [int(x) for x in W.slab_planes(nc[0], S)]
    sph = make_sph(w, with_prev=False)
    sph.sph_set_slabs(planes)
    prev = None
    spread_before, spread_after, multi = [], [], 0
    for k in range(200):
        if k % 20 == 0:
            pos, vel, rho = _state(sph)
            wk = dataclasses.replace(w, pos=pos, vel=vel, rho=rho)
            sph.sph_sort_and_cells()
            sph.sph_build_halos()
            A = compare_structure(sph, wk, planes, prev)
            new = sph.sph_balance_slabs(S)
            assert new == OA.balance_planes(OA.plane_counts(pos, P["dom_min"], P["dom_max"], P["h"]), S)
            sph.sph_build_halos(new)
            A2 = compare_structure(sph, wk, new, prev)
            assert A2["owned"].sum() == w.n
            spread_before.append(A["owned"].max() / A["owned"].mean())
            spread_after.append(A2["owned"].max() / A2["owned"].mean())
            if prev is not None and len(A2["migrants"]):
                multi += np.count_nonzero(np.abs(A2["migrants"][:, 2] - A2["migrants"][:, 3]) > 1)
            # per-slab execution over the new slabs == global pass
            sph.sph_interact()
            ref = sph.sph_download(pos=False, vel=False, rho=False)
            for s in range(S):
                sph.sph_interact_slab(s)
            out = sph.sph_download(pos=False, vel=False, rho=False)
            assert np.array_equal(ref["acc"], out["acc"]) and np.array_equal(ref["drho"], out["drho"])
            planes = new
            prev = owners_by_id(A2, w.n)
            sph.sph_step(w.dt)                            # its sort sees unmoved particles: no migrants
        elif k % 20 == 19:
            # the owners the next re-balance compares with are those of THIS step's sort
            pos, _, _ = _state(sph)
            sph.sph_step(w.dt)
            cx, _, _ = OA.cell_coords(pos, P["dom_min"], P["h"], nc)
            prev = OA.slab_of(cx, planes).astype(np.uint8)
        else:
            sph.sph_step(w.dt)
    assert sph.sph_status() == 0
    assert max(spread_after) < max(spread_before) and spread_after[0] < spread_before[0]
    print("owned max/mean before", np.round(spread_before, 3), "after", np.round(spread_after, 3), "multi", multi)
