"""-m gpu: exact checkpoint / resume ("copied to the host only when saving", L211-212) and
the small boundary fixes of round 2 (single-slab contexts, error text)."""
import numpy as np
import pytest

from paper_1210_1017_b200 import binding as B
from paper_1210_1017_b200 import workloads as W

from gpu_util import make_sph

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("ns", [40, 4])
def test_save_restore_reproduces_the_trajectory_bit_for_bit(ns):
    """7 steps, save, restore into a FRESH context, 7 more == 14 straight (the save falls between
    corrective steps, so the Verlet n-1 state matters)."""
    w = W.dam_break(14, scrambled=True, n_slabs=2)
    w.params = dict(w.params)
    w.params["verlet_ns"] = ns
    a = make_sph(w, with_prev=False)
    for _ in range(14):
        a.sph_step(w.dt)
    ref = a.sph_download()
    ref_m1 = a.sph_download_resume()

    b = make_sph(w, with_prev=False)
    for _ in range(7):
        b.sph_step(w.dt)
    saved = b.sph_download(acc=False, drho=False)
    vel_m1, rho_m1, step = b.sph_download_resume()
    assert step == 7
    b.sph_destroy()

    c = B.Sph(w.params, saved["pos"], saved["vel"], saved["rho"], w.type, max_slabs=16)
    c.sph_set_resume(vel_m1, rho_m1, step)
    assert c.sph_get_view().step_index == 7
    for _ in range(7):
        c.sph_step(w.dt)
    out = c.sph_download()
    for k in ("pos", "vel", "rho", "acc", "drho"):
        assert np.array_equal(out[k].view(np.uint32), ref[k].view(np.uint32)), k
    m1 = c.sph_download_resume()
    assert np.array_equal(m1[0], ref_m1[0]) and np.array_equal(m1[1], ref_m1[1]) and m1[2] == 14
    # without the n-1 state the trajectory differs (the check is not vacuous)
    d = B.Sph(w.params, saved["pos"], saved["vel"], saved["rho"], w.type, max_slabs=16)
    for _ in range(7):
        d.sph_step(w.dt)
    assert not np.array_equal(d.sph_download()["vel"], ref["vel"])
    # resume data is only accepted before the first sort
    with pytest.raises(B.SphError):
        d.sph_set_resume(vel_m1, rho_m1, 7)


def test_single_slab_context_rejects_the_slab_pass():
    """A context created with max_slabs = 1 has no local cell table: sph_interact_slab must refuse
    (round-1 advisor finding: it used to write out of bounds)."""
    w = W.dam_break(10, scrambled=True)
    sph = make_sph(w, max_slabs=1, with_prev=False)
    sph.sph_sort_and_cells()
    sph.sph_build_halos()
    sph.sph_interact()
    ref = sph.sph_download(pos=False, vel=False, rho=False)
    with pytest.raises(B.SphError):
        sph.sph_interact_slab(0)
    out = sph.sph_download(pos=False, vel=False, rho=False)
    assert np.array_equal(ref["acc"], out["acc"]) and sph.sph_status() == 0
    assert sph.sph_last_cuda_error() == ""


def test_nonfinite_velocity_raises_the_flag():
    w = W.dam_break(8, scrambled=True)
    w.vel[5, 1] = np.inf
    sph = make_sph(w, with_prev=False)
    assert sph.sph_status() == -6


def test_fma_peak_is_plausible():
    w = W.dam_break(8)
    sph = make_sph(w, with_prev=False)
    t0, t1 = sph.sph_fma_peak(0, 2048), sph.sph_fma_peak(1, 2048)
    assert 20.0 < t0 < 90.0 and 20.0 < t1 < 90.0, (t0, t1)
