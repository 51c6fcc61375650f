"""-m gpu parity at BASELINE.json's largest configuration (config 3: 31.9 M fluid + 2.06 M boundary
particles, 16 logical x-slabs), in the launch configuration bench.py times: the complete structure
comparison with ORACLE A (numpy lexsort of all 33.9 M keys) and the rates of sampled particles
against ORACLE B, which evaluates each sampled neighbourhood by brute force."""
import numpy as np
import pytest

from oracle import physics as OB
from oracle import structure as OA
from paper_1210_1017_b200 import workloads as W

from gpu_util import compare_structure, make_sph, sampled_rate_errors

pytestmark = pytest.mark.gpu


def test_config3_full_size_structure_and_sampled_rates():
    w = W.dam_break(317, scrambled=True)
    assert w.n == 33910889
    nc = OA.grid_dims(w.params["dom_min"], w.params["dom_max"], w.params["h"])
    planes = W.slab_planes(nc[0], 16)
    sph = make_sph(w)
    sph.sph_set_slabs(planes)
    sph.sph_sort_and_cells()
    sph.sph_build_halos()
    compare_structure(sph, w, planes, None, check_payload=False)
    sph.sph_interact()
    out = sph.sph_download(pos=False, vel=False, rho=False)
    assert sph.sph_status() == 0
    ids = _sample_ids(w, planes, nc, 128, 64, 32, 64)
    assert len(ids) >= 256
    worst_a, scale_a, worst_d, scale_d = sampled_rate_errors(w, out, ids)
    assert scale_a > 0 and scale_d > 0
    assert worst_a <= 1e-4 * scale_a and worst_d <= 1e-4 * scale_d


def _sample_ids(w, planes, nc, n_random, n_wall, n_bound, n_plane):
    """Sampled particle ids: random ones, fluid particles on the faces of the block (their cells also
    hold boundary particles), boundary particles, and fluid particles next to the slab planes."""
    nb = w.notes["nb"]
    nf = w.n_fluid
    dp = w.params["dp"]
    ids = list((W.u01(317, np.arange(n_random), 0) * w.n).astype(np.int64))
    r = (W.u01(318, np.arange(3 * n_wall), 0) * nb).astype(np.int64).reshape(-1, 3)
    for q, (a, b, c) in enumerate(r):
        face = q % 5
        i, j, k = [(0, a, b), (a, 0, b), (a, b, 0), (nb - 1, a, b), (a, nb - 1, b)][face]
        ids.append((i * nb + j) * nb + k)
    ids += list(nf + (W.u01(319, np.arange(n_bound), 0) * (w.n - nf)).astype(np.int64))
    cell = 2.0 * w.params["h"]
    inner = [p for p in planes[1:-1] if 0 < (w.params["dom_min"][0] + p * cell) / dp < nb - 1]
    assert inner
    r = (W.u01(320, np.arange(2 * n_plane), 0) * nb).astype(np.int64).reshape(-1, 2)
    for q, (a, b) in enumerate(r):
        xp = w.params["dom_min"][0] + inner[q % len(inner)] * cell
        i = min(max(int(np.floor(xp / dp)) - (q // len(inner)) % 2, 0), nb - 1)   # lattice layer right / left of the plane
        ids.append((i * nb + a) * nb + b)
    return np.unique(np.asarray(ids, dtype=np.int64))


def test_config2_full_size_structure_and_sampled_rates():
    """BASELINE config 2 (8.8 M particles, 8 slabs) at full size: complete structure comparison and
    the rates of >= 64 sampled particles."""
    w = W.dam_break(200, scrambled=True)
    assert w.n == 8821040
    nc = OA.grid_dims(w.params["dom_min"], w.params["dom_max"], w.params["h"])
    planes = W.slab_planes(nc[0], 8)
    sph = make_sph(w)
    sph.sph_set_slabs(planes)
    sph.sph_sort_and_cells()
    sph.sph_build_halos()
    compare_structure(sph, w, planes, None)
    sph.sph_interact()
    out = sph.sph_download(pos=False, vel=False, rho=False)
    assert sph.sph_status() == 0
    ids = _sample_ids(w, planes, nc, 32, 24, 12, 24)
    assert len(ids) >= 64
    worst_a, scale_a, worst_d, scale_d = sampled_rate_errors(w, out, ids)
    assert scale_a > 0 and scale_d > 0
    assert worst_a <= 1e-4 * scale_a and worst_d <= 1e-4 * scale_d


def test_config3_full_size_ten_steps():
    """BASELINE config 3 (33.9 M particles, 16 slabs rebuilt every step), scrambled start: state after
    10 Verlet steps against ORACLE B stepping the same 10 steps in fp64 (relative L2 <= 1e-3 on r, v,
    rho and on the displacement)."""
    from gpu_util import rel_l2
    w = W.dam_break(317, scrambled=True)
    nc = OA.grid_dims(w.params["dom_min"], w.params["dom_max"], w.params["h"])
    sph = make_sph(w, with_prev=False)
    sph.sph_set_slabs(W.slab_planes(nc[0], 16))
    for _ in range(10):
        sph.sph_step(w.dt)
    out = sph.sph_download(acc=False, drho=False)
    assert sph.sph_status() == 0
    sph.sph_destroy()
    del sph
    p = OB.params_from_workload(w.params)
    s = OB.State(w.pos, w.vel, w.rho, w.type)
    for _ in range(10):
        OB.step(p, s, w.dt, verlet_ns=w.params["verlet_ns"])
    fl = w.type == 0
    assert rel_l2(out["pos"], s.r) <= 1e-3
    assert rel_l2(out["rho"], s.rho) <= 1e-3
    assert rel_l2(out["vel"][fl], s.v[fl]) <= 1e-3
    disp_ref = s.r[fl] - w.pos[fl].astype(np.float64)
    disp = out["pos"][fl].astype(np.float64) - w.pos[fl].astype(np.float64)
    # displacement: 1e-3 relative plus the rounding noise of the fp32 positions themselves (here the
    # two are of the same size: 2.3e-4 and 3.3e-4 m in L2 over 32 M particles)
    from gpu_util import position_rounding_floor
    tol = 1e-3 * np.linalg.norm(disp_ref) + position_rounding_floor(w.pos[fl], 10)
    assert np.linalg.norm(disp - disp_ref) <= tol
    assert np.array_equal(out["pos"][~fl], w.pos[~fl])


def test_config1_full_size_ten_steps():
    """BASELINE config 1 (1.2 M particles, 3 slabs rebuilt every step) at full size: state after 10
    Verlet steps against ORACLE B stepping the same 10 steps in fp64 (north star: relative L2 <= 1e-3)."""
    from gpu_util import rel_l2
    w = W.dam_break(100, scrambled=True, n_slabs=3)
    nc = OA.grid_dims(w.params["dom_min"], w.params["dom_max"], w.params["h"])
    sph = make_sph(w)
    sph.sph_set_slabs(W.slab_planes(nc[0], 3))
    p = OB.params_from_workload(w.params)
    s = OB.State(w.pos, w.vel, w.rho, w.type)
    for _ in range(10):
        sph.sph_step(w.dt)
        OB.step(p, s, w.dt, verlet_ns=w.params["verlet_ns"])
    out = sph.sph_download()
    assert sph.sph_status() == 0
    fl = w.type == 0
    assert rel_l2(out["pos"], s.r) <= 1e-3
    assert rel_l2(out["rho"], s.rho) <= 1e-3
    assert rel_l2(out["vel"][fl], s.v[fl]) <= 1e-3
    disp_ref = s.r[fl] - w.pos[fl].astype(np.float64)
    disp = out["pos"][fl].astype(np.float64) - w.pos[fl].astype(np.float64)
    assert np.linalg.norm(disp - disp_ref) <= 1e-3 * np.linalg.norm(disp_ref)
    assert np.array_equal(out["pos"][~fl], w.pos[~fl])
