"""-m gpu parity at BASELINE.json's largest configuration (config 3: 31.9 M fluid + 2.06 M boundary
particles, 16 logical x-slabs), in the launch configuration bench.py times: the complete structure
comparison with ORACLE A (numpy lexsort of all 33.9 M keys) and the rates of sampled particles
against ORACLE B, which evaluates each sampled neighbourhood by brute force."""
import numpy as np
import pytest

from oracle import physics as OB
from oracle import structure as OA
from paper_1210_1017_b200 import workloads as W

from gpu_util import compare_structure, make_sph

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
    p = OB.params_from_workload(w.params)
    ids = (W.u01(317, np.arange(24), 0) * w.n).astype(np.int64)
    two_h = 2.0 * w.params["h"]
    worst_a = worst_d = scale_a = scale_d = 0.0
    for i in ids:
        pi = w.pos[i].astype(np.float64)
        # cheap pre-selection on x, then the box test on the survivors
        cand = np.nonzero(np.abs(w.pos[:, 0] - np.float32(pi[0])) <= np.float32(two_h * 1.01))[0]
        sub = w.pos[cand].astype(np.float64)
        near = cand[(np.abs(sub - pi) <= two_h * 1.001).all(axis=1)]
        k = int(np.nonzero(near == i)[0][0])
        a, d = OB.rates(p, w.pos[near], w.vel[near], w.rho[near], w.type[near], mode=0)
        if w.type[i] == 0:
            worst_a = max(worst_a, np.abs(out["acc"][i] - a[k]).max())
            scale_a = max(scale_a, np.abs(a[k]).max())
        worst_d = max(worst_d, abs(out["drho"][i] - d[k]))
        scale_d = max(scale_d, abs(d[k]))
    assert scale_a > 0 and scale_d > 0
    assert worst_a <= 1e-4 * scale_a and worst_d <= 1e-4 * scale_d


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
