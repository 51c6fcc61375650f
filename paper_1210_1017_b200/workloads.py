"""Seeded synthetic inputs shared by the oracle tests, the GPU tests and bench.py.

This module holds NO method arithmetic: no cell index, no kernel, no equation of
state, no integrator.  It only lays particles on lattices / in a cube, draws
counter-based random numbers and states the physical parameters of each
configuration named in BASELINE.json ``configs`` (recipe: SURVEY.md section 8(d),
restated in DESIGN.md "Input recipe").  The paper's own runs (dam break with
three obstacles) cannot be reproduced - obstacle geometry and
initial data are not in the paper - so these synthetic inputs stand in for them
with the paper's particle counts (1-8 M per sub-domain, 32 M largest, L360).

Every float handed out is already rounded to fp32 (positions are formed in
fp64 and rounded once), so that the fp64 oracle and the fp32 CUDA path start
from bit-identical inputs.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Optional

import numpy as np

SEED_POS = 1210   # positions / jitter
SEED_STATE = 1017  # scrambled velocities and densities

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _mix64(z: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser on a uint64 array (wrap-around arithmetic)."""
    z = (z + np.uint64(0x9E3779B97F4A7C15)) & _M64
    z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
    z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
    return z ^ (z >> np.uint64(31))


def u01(seed: int, idx: np.ndarray, k: int) -> np.ndarray:
    """Counter-based uniform in [0,1): a pure function of (seed, idx, k).

    u = top 24 bits of mix64(mix64(seed) ^ (idx*4 + k)) * 2^-24   (fp64, exact).
    """
    with np.errstate(over="ignore"):
        s = _mix64(np.array([seed], dtype=np.uint64))[0]
        ctr = (np.asarray(idx, dtype=np.uint64) * np.uint64(4) + np.uint64(k)) & _M64
        z = _mix64(s ^ ctr)
    return (z >> np.uint64(40)).astype(np.float64) * (1.0 / 16777216.0)


def f32(x: float) -> float:
    """Round a python float to fp32 and return it as a python float."""
    return float(np.float32(x))


@dataclass
class Workload:
    name: str
    pos: np.ndarray            # (n,3) float32
    vel: np.ndarray            # (n,3) float32
    rho: np.ndarray            # (n,)  float32
    type: np.ndarray           # (n,)  uint8, 0 fluid, 1 boundary
    params: dict               # physical + grid parameters, all fp32-representable
    dt: float
    n_slabs: int
    n_steps: int
    n_fluid: int
    prev_slab: Optional[np.ndarray] = None   # (n,) uint8 synthetic previous owner, or None
    notes: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.pos.shape[0])


def slab_planes(ncx: int, n_slabs: int) -> np.ndarray:
    """Cell-plane indices of the logical x-slabs: planes[k] = round(k*ncx/S)."""
    return np.array([int(math.floor(k * ncx / n_slabs + 0.5)) for k in range(n_slabs + 1)],
                    dtype=np.int32)


# ----------------------------------------------------------------------------------------
# dam break (BASELINE.json configs[0..3])
# ----------------------------------------------------------------------------------------
_DAM = {  # nb -> (tank Lx, Ly, Lz, slabs, steps)
    16: (0.4, 0.2, 0.3, 1, 10),
    100: (1.6, 0.67, 0.4, 3, 1000),
    200: (1.6, 0.67, 0.4, 8, 500),
    317: (1.6, 0.67, 0.4, 16, 200),
}


def dam_break_params(nb: int, tank=None) -> dict:
    if tank is None:
        tank = _DAM[nb][:3] if nb in _DAM else (0.4, 0.2, 0.3)
    dp = 0.01 if tank[0] == 0.4 else tank[0] / (3.0 * nb)
    h = 1.5 * dp
    H = nb * dp
    g = 9.81
    c0 = 10.0 * math.sqrt(g * H)
    rho0 = 1000.0
    lo = -2.0 * dp - 2.0 * h
    top = max(tank[2], H)
    p = dict(
        dp=f32(dp), h=f32(h), rho0=f32(rho0), c0=f32(c0), alpha=f32(0.01), gamma=7,
        g=(0.0, 0.0, f32(-g)),
        mass_fluid=f32(rho0 * dp ** 3), mass_bound=f32(rho0 * dp ** 3),
        dom_min=(f32(lo), f32(lo), f32(lo)),
        dom_max=(f32(tank[0] + 2 * dp + 2 * h), f32(tank[1] + 2 * dp + 2 * h), f32(top + 2 * dp + 2 * h)),
        verlet_ns=40, kernel=0,
    )
    return p


def dam_break(nb: int = 16, seed: int = SEED_POS, scrambled: bool = False,
              tank=None, n_slabs: Optional[int] = None) -> Workload:
    """3-D dam break: nb^3 fluid lattice block in the corner of an open-top tank
    made of two layers of dynamic boundary particles.

    nb in {16, 100, 200, 317} are BASELINE.json configs[0..3]; other nb give a
    config-0-like tank unless ``tank`` is given.
    """
    if tank is None:
        tank = _DAM[nb][:3] if nb in _DAM else (0.4, 0.2, 0.3)
    S, steps = (_DAM[nb][3], _DAM[nb][4]) if nb in _DAM else (1, 10)
    if n_slabs is not None:
        S = n_slabs
    P = dam_break_params(nb, tank)
    dp = 0.01 if tank[0] == 0.4 else tank[0] / (3.0 * nb)
    nx, ny, nz = (int(math.floor(L / dp + 0.5)) for L in tank)

    # fluid: ids 0..nb^3-1, z fastest
    nf = nb ** 3
    ids = np.arange(nf, dtype=np.int64)
    k = ids % nb
    j = (ids // nb) % nb
    i = ids // (nb * nb)
    pos = np.empty((nf, 3), dtype=np.float64)
    for c, lat in enumerate((i, j, k)):
        jit = (2.0 * u01(seed, ids, c) - 1.0) * 1e-3 * dp
        pos[:, c] = (lat + 0.5) * dp + jit
    fluid = pos.astype(np.float32)
    del pos

    # boundary: lattice sites with index in [-2, n+1] on x,y and [-2, nz-1] on z that
    # are not interior sites (floor + four walls, open top), x-major / z-fastest order.
    bx = np.arange(-2, nx + 2, dtype=np.int64)
    by = np.arange(-2, ny + 2, dtype=np.int64)
    bz = np.arange(-2, nz, dtype=np.int64)
    chunks = []
    # floor slab: all (x, y) for z in {-2,-1}
    X, Y, Z = np.meshgrid(bx, by, bz[:2], indexing="ij")
    floor_sites = np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1)
    # walls: z >= 0, (x,y) on the two-layer rim
    rim_mask = np.ones((bx.size, by.size), dtype=bool)
    rim_mask[2:-2, 2:-2] = False
    rx, ry = np.nonzero(rim_mask)
    zw = bz[2:]
    wall_sites = np.stack([
        np.repeat(bx[rx], zw.size), np.repeat(by[ry], zw.size), np.tile(zw, rx.size)], axis=1)
    sites = np.concatenate([floor_sites, wall_sites], axis=0)
    # canonical order: x-major, z-fastest
    order = np.lexsort((sites[:, 2], sites[:, 1], sites[:, 0]))
    sites = sites[order]
    bound = ((sites.astype(np.float64) + 0.5) * dp).astype(np.float32)
    chunks = [fluid, bound]
    pos32 = np.concatenate(chunks, axis=0)
    n = pos32.shape[0]
    typ = np.zeros(n, dtype=np.uint8)
    typ[nf:] = 1

    vel = np.zeros((n, 3), dtype=np.float32)
    rho = np.full(n, P["rho0"], dtype=np.float32)
    H = nb * dp
    if scrambled:
        allid = np.arange(n, dtype=np.int64)
        vs = 0.1 * math.sqrt(9.81 * H)
        for c in range(3):
            vel[:nf, c] = ((2.0 * u01(SEED_STATE, allid[:nf], c) - 1.0) * vs).astype(np.float32)
        rho = (P["rho0"] * (1.0 + 0.01 * u01(SEED_STATE, allid, 3))).astype(np.float32)

    dt = f32(0.2 * P["h"] / (1.2 * P["c0"]))
    return Workload(
        name=f"dam_break_nb{nb}" + ("_scrambled" if scrambled else ""),
        pos=pos32, vel=vel, rho=rho, type=typ, params=P, dt=dt,
        n_slabs=S, n_steps=steps, n_fluid=nf,
        notes=dict(nb=nb, tank=tank, lattice=(nx, ny, nz), H=H))


# ----------------------------------------------------------------------------------------
# sort / halo microbenchmark (BASELINE.json configs[4])
# ----------------------------------------------------------------------------------------
def uniform_cube(n: int, seed: int = SEED_POS, n_slabs: int = 8, chunk: int = 1 << 24) -> Workload:
    """n particles uniform in [0,1)^3, ids in generation order (random cell keys), cell
    size 2h with a mean of ~30 neighbours inside the 2h sphere, velocities U(-1,1).

    ``prev_slab`` is a synthetic previous owner: the k/S-slab of x shifted by U(-0.2,0.2)*2h,
    so a few per cent of the particles show up as migrants, about half of them in each direction
    (labels 1 and 2 of PAPER.md L264).
    """
    two_h = (90.0 / (4.0 * math.pi * n)) ** (1.0 / 3.0)
    h = 0.5 * two_h
    pos = np.empty((n, 3), dtype=np.float32)
    vel = np.empty((n, 3), dtype=np.float32)
    prev = np.empty(n, dtype=np.uint8)
    for a in range(0, n, chunk):
        b = min(n, a + chunk)
        ids = np.arange(a, b, dtype=np.int64)
        for c in range(3):
            pos[a:b, c] = u01(seed, ids, c).astype(np.float32)
        for c in range(3):
            vel[a:b, c] = (2.0 * u01(SEED_STATE, ids, c) - 1.0).astype(np.float32)
        xs = pos[a:b, 0].astype(np.float64) + 0.2 * two_h * (2.0 * u01(SEED_STATE, ids, 3) - 1.0)
        prev[a:b] = np.clip(np.floor(xs * n_slabs), 0, n_slabs - 1).astype(np.uint8)
    # fp32 rounding can push u < 1 up to exactly 1.0f; keep the cube half-open
    np.minimum(pos, np.float32(np.nextafter(np.float32(1.0), np.float32(0.0))), out=pos)
    rho0 = 1000.0
    dp = (1.0 / n) ** (1.0 / 3.0)
    P = dict(
        dp=f32(dp), h=f32(h), rho0=f32(rho0), c0=f32(30.0), alpha=f32(0.01), gamma=7,
        g=(0.0, 0.0, f32(-9.81)),
        mass_fluid=f32(rho0 / n), mass_bound=f32(rho0 / n),
        dom_min=(0.0, 0.0, 0.0), dom_max=(1.0, 1.0, 1.0),
        verlet_ns=40, kernel=0,
    )
    return Workload(
        name=f"uniform_cube_{n}", pos=pos, vel=vel,
        rho=np.full(n, P["rho0"], dtype=np.float32), type=np.zeros(n, dtype=np.uint8),
        params=P, dt=f32(0.2 * P["h"] / (1.2 * P["c0"])), n_slabs=n_slabs, n_steps=1,
        n_fluid=n, prev_slab=prev, notes=dict(two_h=two_h))


# ----------------------------------------------------------------------------------------
# small structured inputs used by the oracle pins and edge-case parity tests
# ----------------------------------------------------------------------------------------
def lattice_block(nx: int, ny: int, nz: int, dp: float, origin=(0.0, 0.0, 0.0)) -> np.ndarray:
    """Unjittered cubic lattice, sites (i+1/2)*dp + origin, z fastest; float64 (n,3)."""
    i, j, k = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij")
    p = np.stack([i.ravel(), j.ravel(), k.ravel()], axis=1).astype(np.float64)
    return (p + 0.5) * dp + np.asarray(origin, dtype=np.float64)


def random_box(n: int, box, seed: int = SEED_POS) -> np.ndarray:
    """n points uniform in [0,box) per axis; float64 (n,3)."""
    ids = np.arange(n, dtype=np.int64)
    return np.stack([u01(seed, ids, c) * box[c] for c in range(3)], axis=1)
