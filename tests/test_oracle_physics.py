"""Pins for ORACLE B (oracle/sph_physics.c): closed forms, invariants, brute force.

Each test is chosen so that a plausible mistake in the oracle (a dropped term, a wrong
sign or index, p/rho instead of p/rho^2, a transposed r_ij) fails at least one of them.
"""
import math
import os

import numpy as np
import pytest

from oracle import physics as OB
from paper_1210_1017_b200 import workloads as W


def _golden(path):
    out = {}
    with open(path) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                k, v = line.split()
                out[k] = float(v)
    return out


# ---------------------------------------------------------------- kernel
@pytest.mark.parametrize("kernel", [0, 1])
def test_kernel_unit_integral_and_support(kernel):
    h = 0.37
    p = OB.make_params(h=h, kernel=kernel)
    # composite Simpson on [0, 2h]; both kernels are piecewise polynomials
    m = 4000
    r = np.linspace(0.0, 2.0 * h, m + 1)
    f = np.array([OB.W(p, x) * 4.0 * math.pi * x * x for x in r])
    integral = (r[1] - r[0]) / 3.0 * (f[0] + f[-1] + 4.0 * f[1:-1:2].sum() + 2.0 * f[2:-1:2].sum())
    assert abs(integral - 1.0) < 1e-6
    assert OB.W(p, 2.0 * h) == 0.0 and OB.W(p, 2.5 * h) == 0.0
    assert OB.F(p, 2.0 * h) == 0.0
    w = [OB.W(p, x) for x in np.linspace(0, 2 * h, 200)]
    assert all(a >= b for a, b in zip(w[:-1], w[1:]))          # monotone decreasing
    assert w[0] > 0


@pytest.mark.parametrize("kernel", [0, 1])
def test_kernel_gradient_matches_finite_difference(kernel):
    h = 0.8
    p = OB.make_params(h=h, kernel=kernel)
    for r in (0.05, 0.3, 0.79, 0.81, 1.2, 1.59):
        e = 1e-6
        dW = (OB.W(p, r + e) - OB.W(p, r - e)) / (2 * e)
        assert abs(OB.F(p, r) * r - dW) < 1e-7 * max(1.0, abs(dW))
        assert OB.F(p, r) < 0.0


# ---------------------------------------------------------------- EOS (L112)
def test_tait_eos():
    p = OB.make_params(h=1.0, rho0=1000.0, c0=37.0, gamma=7.0)
    assert OB.pressure(p, 1000.0) == 0.0
    e = 1e-3
    slope = (OB.pressure(p, 1000.0 + e) - OB.pressure(p, 1000.0 - e)) / (2 * e)
    assert abs(slope - 37.0 ** 2) < 1e-4 * 37.0 ** 2            # c0^2 = dp/drho at rho0
    assert abs(OB.sound_speed(p, 1000.0) - 37.0) < 1e-12
    # c(rho)^2 is the local slope of the EOS
    rho = 1030.0
    slope = (OB.pressure(p, rho + e) - OB.pressure(p, rho - e)) / (2 * e)
    assert abs(OB.sound_speed(p, rho) ** 2 - slope) < 1e-5 * slope


# ---------------------------------------------------------------- two particles, by hand
def test_two_particle_closed_forms(golden_dir):
    G = _golden(os.path.join(golden_dir, "two_particle_closed_forms.txt"))
    p = OB.make_params(h=1.0, rho0=1000.0, c0=10.0, alpha=0.5, gamma=7.0, g=(0, 0, 0), mass_fluid=3.0)
    assert abs(OB.F(p, 1.0) - G["F"]) < 1e-14
    r = [[0, 0, 0], [1, 0, 0]]
    typ = [0, 0]
    for mode in (0, 1):
        acc, drho = OB.rates(p, r, [[2, 0, 0], [0, 0, 0]], [1000, 1000], typ, mode=mode)
        assert abs(drho[0] - G["A_drho"]) < 1e-13 and abs(drho[1] - G["A_drho"]) < 1e-13
        assert abs(acc[0, 0] - G["A_aix"]) < 1e-15 and abs(acc[1, 0] + G["A_aix"]) < 1e-15
        assert (acc[:, 1:] == 0).all()
        # receding pair: no viscosity, and rho = rho0 => p = 0 => no force at all
        acc, drho = OB.rates(p, r, [[-2, 0, 0], [0, 0, 0]], [1000, 1000], typ, mode=mode)
        assert (acc == 0).all() and abs(drho[0] + G["A_drho"]) < 1e-13
        # pressure only
        acc, drho = OB.rates(p, r, np.zeros((2, 3)), [1010, 1010], typ, mode=mode)
        assert abs(acc[0, 0] - G["B_aix"]) < 1e-14 and abs(acc[1, 0] + G["B_aix"]) < 1e-14
        assert (drho == 0).all()
    # beyond the support (r = 2h exactly, and further) nothing interacts; coincident skipped
    acc, drho = OB.rates(p, [[0, 0, 0], [2, 0, 0]], [[2, 0, 0], [0, 0, 0]], [1010, 1010], typ, mode=0)
    assert (acc == 0).all() and (drho == 0).all()
    acc, drho = OB.rates(p, [[0, 0, 0], [0, 0, 0]], [[2, 0, 0], [0, 0, 0]], [1010, 1010], typ, mode=0)
    assert np.isfinite(acc).all() and (acc == 0).all() and (drho == 0).all()
    # a boundary particle feels the density rate but has zero acceleration (L116)
    acc, drho = OB.rates(p, r, [[2, 0, 0], [0, 0, 0]], [1000, 1000], [1, 0], mode=0)
    assert (acc[0] == 0).all() and abs(drho[0] - G["A_drho"]) < 1e-13 and acc[1, 0] > 0
    # gravity is added to fluid particles only
    p.g[2] = -9.81
    acc, _ = OB.rates(p, [[0, 0, 0], [5, 0, 0]], np.zeros((2, 3)), [1000, 1000], [0, 1], mode=0)
    assert acc[0, 2] == -9.81 and acc[1, 2] == 0.0


# ---------------------------------------------------------------- lattice field tests
def _lattice(nside, dp):
    r = W.lattice_block(nside, nside, nside, dp)
    centre = (nside // 2 * nside + nside // 2) * nside + nside // 2
    return r, centre


@pytest.mark.parametrize("kernel", [0, 1])
def test_continuity_is_minus_rho_div_v(kernel):
    """Eq. (7) must discretise Eq. (1) D rho/Dt = -rho div v (L55): linear field v = A r.
    With h = 2.5 dp the lattice sum is within 2e-3 of the continuum value."""
    dp, nside = 0.1, 13
    h = 2.5 * dp
    r, c = _lattice(nside, dp)
    A = np.array([[0.3, 0.1, -0.2], [0.05, -0.7, 0.4], [0.6, -0.1, 0.9]])
    v = r @ A.T
    rho0 = 1000.0
    p = OB.make_params(h=h, rho0=rho0, g=(0, 0, 0), mass_fluid=rho0 * dp ** 3, kernel=kernel)
    n = r.shape[0]
    acc, drho = OB.rates(p, r, v, np.full(n, rho0), np.zeros(n, np.uint8))
    expect = -rho0 * np.trace(A)
    tol = 2e-3 if kernel == 0 else 5e-3          # the C2 cubic spline converges more slowly
    assert abs(drho[c] - expect) < tol * abs(expect)
    # pure expansion => density falls
    acc, drho = OB.rates(p, r, r * 1.0, np.full(n, rho0), np.zeros(n, np.uint8))
    assert drho[c] < 0


@pytest.mark.parametrize("kernel", [0, 1])
def test_pressure_gradient_form_p_over_rho_squared(kernel):
    """Eq. (9) must discretise Eq. (2) Dv/Dt = -(1/rho) grad p + g (L57).  Prescribed
    p = G z at rho = rho0: a - g = -G/rho0 z^.  The printed p/rho form (reading A2) would
    be off by a factor rho0 = 1000."""
    dp, nside = 0.1, 13
    h = 2.5 * dp
    r, c = _lattice(nside, dp)
    rho0, G = 1000.0, 2500.0
    g = (0.0, 0.0, -9.81)
    p = OB.make_params(h=h, rho0=rho0, g=g, mass_fluid=rho0 * dp ** 3, kernel=kernel)
    n = r.shape[0]
    acc, drho = OB.rates(p, r, np.zeros((n, 3)), np.full(n, rho0), np.zeros(n, np.uint8),
                         p_override=G * r[:, 2])
    a = acc[c] - np.array(g)
    tol = 2e-3 if kernel == 0 else 5e-3
    assert abs(a[2] - (-G / rho0)) < tol * G / rho0
    assert abs(a[0]) < 1e-9 and abs(a[1]) < 1e-9
    assert (drho == 0).all()
    # gradient along x picks the x component (index / transposition check)
    acc, _ = OB.rates(p, r, np.zeros((n, 3)), np.full(n, rho0), np.zeros(n, np.uint8),
                      p_override=G * r[:, 0])
    a = acc[c] - np.array(g)
    assert abs(a[0] - (-G / rho0)) < tol * G / rho0 and abs(a[2]) < 1e-9


def test_uniform_compression_viscosity_is_repulsive():
    """Pi_ij > 0 for every approaching pair (L112): under v = -r the viscous term opposes
    the compression; with p = 0 (rho = rho0) it is the only force: a points outward from a
    denser side, i.e. for an off-centre particle next to a void it decelerates it."""
    dp, nside = 0.1, 9
    h = 1.5 * dp
    r, c = _lattice(nside, dp)
    rho0 = 1000.0
    n = r.shape[0]
    p0 = OB.make_params(h=h, rho0=rho0, c0=20.0, alpha=0.0, g=(0, 0, 0), mass_fluid=rho0 * dp ** 3)
    p1 = OB.make_params(h=h, rho0=rho0, c0=20.0, alpha=0.3, g=(0, 0, 0), mass_fluid=rho0 * dp ** 3)
    ctr = r[c]
    v = -(r - ctr)
    a0, _ = OB.rates(p0, r, v, np.full(n, rho0), np.zeros(n, np.uint8))
    a1, _ = OB.rates(p1, r, v, np.full(n, rho0), np.zeros(n, np.uint8))
    assert (a0 == 0).all()                       # no pressure, no viscosity => nothing
    corner = 0                                   # particle at the block corner moves inward (+,+,+)
    assert (a1[corner] < 0).all()                # viscous force pushes it back outward
    # same field reversed (expansion): receding pairs => no viscosity anywhere
    a2, _ = OB.rates(p1, r, -v, np.full(n, rho0), np.zeros(n, np.uint8))
    assert (a2 == 0).all()


# ---------------------------------------------------------------- conservation
def _periodic_case(kernel=0):
    n, L = 700, (1.0, 0.9, 0.8)
    r = W.random_box(n, L, seed=11)
    ids = np.arange(n)
    v = np.stack([2 * W.u01(5, ids, c) - 1 for c in range(3)], axis=1)
    rho = 1000.0 * (1 + 0.02 * W.u01(5, ids, 3))
    h = 0.11
    p = OB.make_params(h=h, rho0=1000.0, c0=30.0, alpha=0.2, g=(0, 0, 0), mass_fluid=1.3,
                       kernel=kernel, periodic=(1, 1, 1), box_min=(0, 0, 0), box_len=L)
    return p, r, v, rho, np.zeros(n, np.uint8)


@pytest.mark.parametrize("kernel", [0, 1])
def test_pair_antisymmetry_conserves_linear_momentum(kernel):
    p, r, v, rho, typ = _periodic_case(kernel)
    acc, drho = OB.rates(p, r, v, rho, typ, mode=0)
    scale = np.abs(acc).sum(axis=0)
    assert (np.abs(acc.sum(axis=0)) < 1e-11 * scale).all()
    assert np.abs(acc).max() > 0
    # exact mass conservation: masses are constants, particle count unchanged by a step
    s = OB.State(r, v, rho, typ)
    OB.step(p, s, 1e-4)
    assert s.n == len(rho)


def test_cell_list_equals_brute_force_bitwise():
    p, r, v, rho, typ = _periodic_case()
    a0, d0 = OB.rates(p, r, v, rho, typ, mode=0)
    a1, d1 = OB.rates(p, r, v, rho, typ, mode=1)
    assert (a0 == a1).all() and (d0 == d1).all()
    # non-periodic, with boundary particles and gravity
    w = W.dam_break(6, scrambled=True)
    q = OB.params_from_workload(w.params)
    a0, d0 = OB.rates(q, w.pos, w.vel, w.rho, w.type, mode=0)
    a1, d1 = OB.rates(q, w.pos, w.vel, w.rho, w.type, mode=1)
    assert (a0 == a1).all() and (d0 == d1).all()
    assert np.abs(d0).max() > 0 and (a0[w.type == 1] == 0).all()


# ---------------------------------------------------------------- integrator (L150, reading A7)
def test_verlet_free_fall_and_fixed_boundary():
    g = 9.81
    p = OB.make_params(h=0.1, g=(0, 0, -g))
    # two far-apart particles: one fluid, one boundary.  The boundary particle CARRIES a velocity (an
    # "externally imposed" one, L116): integrating it would move it, so the branch is visible
    s = OB.State([[0, 0, 10.0], [50, 0, 0]], [[0.3, 0, 0], [0.2, 0, 0]], [1000, 1000], [0, 1])
    dt, ns = 1e-3, 4
    for n in range(1, 11):                       # exercises corrective (n % 4 == 0) and leapfrog steps
        OB.step(p, s, dt, verlet_ns=ns, mode=0)
        t = n * dt
        assert abs(s.r[0, 2] - (10.0 - 0.5 * g * t * t)) < 1e-12
        assert abs(s.v[0, 2] + g * t) < 1e-12
        assert abs(s.r[0, 0] - 0.3 * t) < 1e-12
        # L116: "the integration update for position and velocity is not performed"
        assert (s.r[1] == [50, 0, 0]).all() and (s.v[1] == [0.2, 0, 0]).all()
    assert s.rho[0] == 1000 and s.rho[1] == 1000


def test_boundary_particle_density_evolves_but_position_and_velocity_do_not():
    """boundary particles "satisfy the same equations as the fluid particles" except that
    "the integration update for position and velocity is not performed" - so next to approaching fluid a
    moving wall particle's density follows its continuity rate (Eq. 7) while r and v keep their bits.
    The rate is pinned by hand: d rho_b/dt = m_f (v_b - v_f) . grad_b W(r_b - r_f), Wendland C2 in 3-D,
    dW/dr = -(105 / (16 pi h^5)) r (1 - r/2h)^3  (written out here, not taken from the oracle)."""
    h, m = 0.1, 0.7
    p = OB.make_params(h=h, g=(0, 0, -9.81), mass_fluid=m, mass_bound=m)
    rb, rf = np.array([0.0, 0.0, 0.0]), np.array([0.12, 0.0, 0.05])
    vb, vf = np.array([0.2, -0.1, 0.0]), np.array([-1.0, 0.0, 0.5])
    s = OB.State([rb, rf], [vb, vf], [1000.0, 1000.0], [1, 0])
    d = rb - rf
    r = float(np.linalg.norm(d))
    dWdr = -(105.0 / (16.0 * np.pi * h ** 5)) * r * (1.0 - r / (2 * h)) ** 3
    drho_b = m * float(np.dot(vb - vf, d / r)) * dWdr
    assert abs(drho_b) > 1.0
    dt = 1e-4
    rho = [1000.0]
    for n in range(3):                           # step 0 is one-sided, steps 1, 2 use rho_m1 + 2 dt rate
        rates_a, rates_d = OB.rates(p, s.r, s.v, s.rho, s.type, mode=0)
        if n == 0:
            assert abs(rates_d[0] - drho_b) <= 1e-12 * abs(drho_b)
        assert (rates_a[0] == 0).all()           # no acceleration is kept for a boundary particle
        rho.append((rho[-1] if n == 0 else rho[-2]) + (1 if n == 0 else 2) * dt * rates_d[0])
        OB.step(p, s, dt, verlet_ns=40, mode=0)
        assert (s.r[0] == rb).all() and (s.v[0] == vb).all()            # bit-unchanged
        assert abs(s.rho[0] - rho[-1]) <= 1e-12 * 1000.0 and s.rho[0] != 1000.0
        assert (s.r[1] != rf).any() and (s.v[1] != vf).any()            # the fluid particle does move


def test_verlet_uses_two_step_form_between_corrections():
    """v+ = v_m1 + 2 dt a on ordinary steps, v + dt a on corrective ones: feed a state with
    v_m1 != v and check which branch was taken."""
    s = OB.State([[0, 0, 0]], [[1.0, 0, 0]], [1000], [0])
    s.v_m1[:] = [[0.5, 0, 0]]
    s.rho_m1[:] = [990.0]
    acc = np.array([[2.0, 0, 0]])
    drho = np.array([10.0])
    import ctypes as C
    dp = C.POINTER(C.c_double)
    for corrective, v_exp, rho_exp in ((0, 0.5 + 2 * 0.1 * 2.0, 990.0 + 2 * 0.1 * 10.0),
                                       (1, 1.0 + 0.1 * 2.0, 1000.0 + 0.1 * 10.0)):
        t = OB.State(s.r, s.v, s.rho, s.type)
        t.v_m1[:] = s.v_m1
        t.rho_m1[:] = s.rho_m1
        OB.lib().orc_verlet(1, t.r.ctypes.data_as(dp), t.v.ctypes.data_as(dp), t.rho.ctypes.data_as(dp),
                            t.v_m1.ctypes.data_as(dp), t.rho_m1.ctypes.data_as(dp), t.type.ctypes.data,
                            acc.ctypes.data_as(dp), drho.ctypes.data_as(dp), 0.1, corrective)
        assert abs(t.v[0, 0] - v_exp) < 1e-15 and abs(t.rho[0] - rho_exp) < 1e-12
        assert abs(t.r[0, 0] - (0.1 * 1.0 + 0.5 * 0.01 * 2.0)) < 1e-15
        assert t.v_m1[0, 0] == 1.0 and t.rho_m1[0] == 1000.0


# ---------------------------------------------------------------- whole step
def test_hydrostatic_column_bottom_pressure():
    """A laterally periodic water column resting on dynamic boundary particles settles to
    p(bottom) = rho0 g depth within 2 % (time-averaged)."""
    dp = 0.02
    h = 1.5 * dp
    nx = ny = 6                      # 6 dp = 4h wide: two 2h-cells per periodic direction ... use 9
    nx = ny = 9
    nzf, nzb = 30, 3
    g, rho0 = 9.81, 1000.0
    Hc = nzf * dp
    c0 = 10.0 * math.sqrt(g * Hc)
    B = c0 * c0 * rho0 / 7.0
    rb = W.lattice_block(nx, ny, nzb, dp, origin=(0, 0, -nzb * dp))
    rf = W.lattice_block(nx, ny, nzf, dp)
    r = np.concatenate([rf, rb])
    typ = np.concatenate([np.zeros(len(rf), np.uint8), np.ones(len(rb), np.uint8)])
    depth = np.clip(Hc - r[:, 2], 0.0, None)
    rho = rho0 * (1.0 + rho0 * g * depth / B) ** (1.0 / 7.0)     # hydrostatic start (inverse Tait)
    p = OB.make_params(h=h, rho0=rho0, c0=c0, alpha=0.5, g=(0, 0, -g), mass_fluid=rho0 * dp ** 3,
                       periodic=(1, 1, 0), box_min=(0, 0, 0), box_len=(nx * dp, ny * dp, 1.0))
    s = OB.State(r, np.zeros_like(r), rho, typ)
    dt = 0.2 * h / (1.2 * c0)
    # bottom fluid layer (k = 0) sits at depth Hc - dp/2
    layer = np.nonzero((typ == 0) & (np.abs(r[:, 2] - 0.5 * dp) < 1e-9))[0]
    mid = np.nonzero((typ == 0) & (np.abs(r[:, 2] - 10.5 * dp) < 1e-9))[0]
    nsteps, tail = 1500, 700
    pb, pm = [], []
    for n in range(nsteps):
        OB.step(p, s, dt, verlet_ns=40)
        if n >= nsteps - tail:
            pb.append(np.mean([OB.pressure(p, x) for x in s.rho[layer]]))
            pm.append(np.mean([OB.pressure(p, x) for x in s.rho[mid]]))
    assert np.isfinite(s.r).all()
    z_b = s.r[layer, 2].mean()
    z_m = s.r[mid, 2].mean()
    top = s.r[typ == 0, 2].max() + 0.5 * dp
    assert abs(np.mean(pb) - rho0 * g * (top - z_b)) < 0.02 * rho0 * g * Hc
    assert abs(np.mean(pm) - rho0 * g * (top - z_m)) < 0.02 * rho0 * g * Hc
    # the column stays a column (no lateral drift, little vertical motion)
    assert np.abs(s.r[typ == 0, :2] - rf[:, :2]).max() < 0.05 * dp
    assert np.abs(s.r[typ == 0, 2] - rf[:, 2]).max() < 0.5 * dp


# ---- variable time step (reading A8b; L150, L222) ---------------------------------------------
def test_time_step_two_particles_by_hand():
    """h = 0.1, eta^2 = 0.01 h^2 = 1e-4.  Particles 0.15 apart along x approaching at 1 m/s:
    mu = h |v.r| / (r^2 + eta^2) = 0.1 * 0.15 / (0.0225 + 0.0001) = 0.015 / 0.0226.
    dt_cv = h / (c0 + mu) with rho = rho0; dt_f = sqrt(h / 9.81) from the larger acceleration."""
    p = OB.make_params(h=0.1, c0=10.0)
    r = np.array([[0, 0, 0], [0.15, 0, 0.0]])
    v = np.array([[0, 0, 0], [-1.0, 0, 0]])
    rho = np.array([1000.0, 1000.0])
    acc = np.array([[0, 0, -9.81], [0, 0, -2.0]])
    o = OB.time_step(p, r, v, rho, np.zeros(2, np.uint8), acc, cfl=0.2)
    mu = 0.015 / 0.0226
    assert np.allclose(o["mu"], [mu, mu], rtol=1e-14)
    assert abs(o["dt_cv"] - 0.1 / (10.0 + mu)) < 1e-16
    assert abs(o["dt_f"] - np.sqrt(0.1 / 9.81)) < 1e-16
    assert abs(o["dt"] - 0.2 * 0.1 / (10.0 + mu)) < 1e-16
    # receding pairs count with their magnitude too (|mu|)
    o2 = OB.time_step(p, r, -v, rho, np.zeros(2, np.uint8), acc, cfl=0.2)
    assert np.allclose(o2["mu"], o["mu"], rtol=1e-14)
    # a boundary particle's acceleration does not limit the step; beyond 2h there is no pair
    o3 = OB.time_step(p, r * 2.0, v, rho, np.array([1, 0], np.uint8), acc, cfl=0.2)
    assert (o3["mu"] == 0).all() and abs(o3["dt_f"] - np.sqrt(0.1 / 2.0)) < 1e-16
    assert abs(o3["dt_cv"] - 0.1 / 10.0) < 1e-18


def test_time_step_uniform_expansion_on_a_lattice_and_the_cut_off():
    """dp = 1, h = 1.5 (4h^2 = 9 exactly), v = A r: v_ij.r_ij = A r^2, so mu grows with r and the
    maximum sits at the farthest neighbour: |n|^2 = 8 inside the support, the 30 lattice points at
    |n|^2 = 9 lie exactly ON the edge (excluded by r < 2h, included by cut > 1): this is the
    discontinuity a bracketing comparison of an fp32 implementation has to allow for."""
    n1 = 7
    g = np.arange(n1, dtype=np.float64)
    r = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    A = 0.3
    v = A * r
    rho = np.full(len(r), 1000.0)
    p = OB.make_params(h=1.5, c0=20.0)
    acc = np.zeros_like(r)
    centre = (3 * n1 + 3) * n1 + 3
    o = OB.time_step(p, r, v, rho, np.zeros(len(r), np.uint8), acc)
    assert abs(o["mu"][centre] - 1.5 * A * 8.0 / (8.0 + 0.0225)) < 1e-14
    o = OB.time_step(p, r, v, rho, np.zeros(len(r), np.uint8), acc, cut=1.0 + 1e-9)
    assert abs(o["mu"][centre] - 1.5 * A * 9.0 / (9.0 + 0.0225)) < 1e-14
    assert o["dt_f"] == np.inf


def test_time_step_per_slab_minimum_is_the_global_one():
    """L222: every sub-domain finds its own dt_k; the step uses the minimum."""
    rng = np.random.default_rng(5)
    n = 400
    r = rng.random((n, 3)) * 0.5
    v = rng.normal(size=(n, 3))
    rho = 1000.0 * (1 + 0.01 * rng.random(n))
    typ = (rng.random(n) < 0.2).astype(np.uint8)
    acc = rng.normal(size=(n, 3)) * 10
    p = OB.make_params(h=0.05, c0=30.0)
    slab = np.minimum((r[:, 0] / 0.5 * 4).astype(np.int64), 3)
    o = OB.time_step(p, r, v, rho, typ, acc, cfl=0.2, slab_of=slab, n_slabs=4)
    dt_k = 0.2 * np.minimum(np.sqrt(0.05 / o["amax_slab"]), 0.05 / o["smax_slab"])
    assert abs(dt_k.min() - o["dt"]) < 1e-18
    # brute-force restatement of the maxima in numpy
    fl = typ == 0
    assert abs(o["amax_slab"].max() - np.linalg.norm(acc[fl], axis=1).max()) < 1e-12
    d = r[:, None, :] - r[None, :, :]
    r2 = (d ** 2).sum(-1)
    dot = ((v[:, None, :] - v[None, :, :]) * d).sum(-1)
    mu = np.where((r2 < 4 * 0.05 ** 2) & (r2 > 0), np.abs(0.05 * dot / (r2 + 0.01 * 0.05 ** 2)), 0.0).max(1)
    assert np.allclose(mu, o["mu"], rtol=1e-12, atol=0)
