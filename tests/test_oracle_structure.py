"""Pins for ORACLE A (oracle/structure.py): what the paper prints, brute force, closed forms."""
import math
import os

import numpy as np

from oracle import physics as OB
from oracle import structure as OA
from paper_1210_1017_b200 import workloads as W


def _read_rows(path):
    rows = []
    with open(path) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                rows.append([int(x) for x in line.split()])
    return rows


def test_paper_worked_example(golden_dir):
    """radix sort of ids by halo label; stable, ids ascending inside a label."""
    halo_in, id_in, halo_out, id_out = _read_rows(os.path.join(golden_dir, "paper_halo_sort_example.txt"))
    order = OA.sort_by_label(halo_in, id_in)
    assert [halo_in[k] for k in order] == halo_out
    assert [id_in[k] for k in order] == id_out
    # history-free: the same result from a scrambled presentation of the same (label, id) pairs
    perm = [5, 2, 7, 0, 3, 6, 1, 4]
    order2 = OA.sort_by_label([halo_in[k] for k in perm], [id_in[k] for k in perm])
    assert [id_in[perm[k]] for k in order2] == id_out


def test_cell_label_hand_placed():
    """Exactly representable coordinates: h = 0.25 => 2h cells of side 0.5 on [-1,1)^3 => 4^3 cells."""
    dom_min, dom_max, h = (-1.0, -1.0, -1.0), (1.0, 1.0, 1.0), 0.25
    nc = OA.grid_dims(dom_min, dom_max, h)
    assert nc == (4, 4, 4)
    pos = np.array([
        [0.25, -0.75, 0.9],     # (2,0,3)
        [0.0, 0.0, 0.0],        # on three faces -> belongs to the upper cell (2,2,2)
        [-1.0, -1.0, -1.0],     # domain corner (0,0,0)
        [5.0, -3.0, 0.1],       # outside -> clamped (3,0,2)
        [0.999, 0.4999, -0.5],  # (3,2,1): -0.5 is a face -> cell 1
    ], dtype=np.float32)
    cx, cy, cz = OA.cell_coords(pos, dom_min, h, nc)
    assert list(zip(cx, cy, cz)) == [(2, 0, 3), (2, 2, 2), (0, 0, 0), (3, 0, 2), (3, 2, 1)]
    cell = OA.cell_index(cx, cy, cz, nc)
    assert list(cell) == [(2 * 4 + 0) * 4 + 3, 42, 0, (3 * 4 + 0) * 4 + 2, (3 * 4 + 2) * 4 + 1]


def test_grid_dims_configs():
    """2h = 3dp cells; config 0 tank 0.4x0.2x0.3 with a 5dp margin each side: 50/25/35 dp."""
    w = W.dam_break(16)
    nc = OA.grid_dims(w.params["dom_min"], w.params["dom_max"], w.params["h"])
    # hand derivation: extent = tank + 2 (2 dp + 2h) = tank + 10 dp, cell = 3 dp.  The number of cells
    # is ceil(extent / cell); where the real quotient is an integer the fp32 rounding of the
    # parameters decides between q and q + 1 (both listed), elsewhere the value is forced.
    hand = {  # nb: per axis (extent in dp, forced value or the two candidates)
        16: ((50.0, (17,)), (30.0, (10, 11)), (40.0, (14,))),                      # 16.67, 10, 13.33
        100: ((310.0, (104,)), (135.625, (46,)), (110.0, (37,))),                 # 103.33, 45.2, 36.67
        200: ((610.0, (204,)), (261.25, (88,)), (210.0, (70, 71))),               # 203.33, 87.08, 70
        317: ((961.0, (321,)), (408.23125, (137,)), (327.0, (109, 110))),         # 320.33, 136.08, 109
    }
    exact = {16: (17, 11, 14), 100: (104, 46, 37), 200: (204, 88, 70), 317: (321, 137, 110)}
    for nb, axes in hand.items():
        P = W.dam_break_params(nb)
        got = OA.grid_dims(P["dom_min"], P["dom_max"], P["h"])
        for k, (ext_dp, allowed) in enumerate(axes):
            q = ext_dp / 3.0
            if abs(q - round(q)) > 1e-6:
                assert allowed == (math.ceil(q),)
            assert got[k] in allowed, (nb, k, got)
        assert got == exact[nb]
    assert nc == exact[16]
    # every particle of the config lies strictly inside the grid (no clamping active)
    inv = 1.0 / (2.0 * w.params["h"])
    t = (w.pos.astype(np.float64) - np.array(w.params["dom_min"])) * inv
    assert (t > 0).all() and (t < np.array(nc)).all()


def _brute_structure(pos32, ids, dom_min, dom_max, h, planes, prev):
    """Pure-python loops, no numpy sorting/searching - the set definitions."""
    nc = OA.grid_dims(dom_min, dom_max, h)
    inv = np.float32(1.0) / (np.float32(2.0) * np.float32(h))
    n = len(ids)
    cells, cxs = [], []
    for p in pos32:
        c = []
        for k in range(3):
            t = np.float32(np.float32(p[k]) - np.float32(dom_min[k])) * inv
            c.append(min(max(int(math.floor(float(t))), 0), nc[k] - 1))
        cells.append((c[0] * nc[1] + c[1]) * nc[2] + c[2])
        cxs.append(c[0])
    S = len(planes) - 1
    slab = [max(s for s in range(S) if planes[s] <= cx) for cx in cxs]
    order = sorted(range(n), key=lambda k: (cells[k], ids[k]))
    ncells = nc[0] * nc[1] * nc[2]
    begin = [sum(1 for k in range(n) if cells[k] < c) for c in range(ncells + 1)]
    end = [sum(1 for k in range(n) if cells[k] <= c) for c in range(ncells + 1)]
    halo = []
    for s in range(S):
        L = [ids[k] for k in order if s > 0 and cxs[k] == planes[s] - 1]
        R = [ids[k] for k in order if s < S - 1 and cxs[k] == planes[s + 1]]
        halo.append((L, R))
    hl = []
    for k in range(n):
        s = slab[k]
        lab = 0
        if s > 0 and cxs[k] == planes[s]:
            lab = 1
        if s < S - 1 and cxs[k] == planes[s + 1] - 1:
            lab = 2
        ml = 0
        if prev is not None:
            ml = 1 if slab[k] < prev[k] else (2 if slab[k] > prev[k] else 0)
        hl.append(lab + 4 * ml)
    kw = [(hl[k] << 28) + cells[k] for k in order]
    mig = [(ids[k], rank, prev[k], slab[k]) for rank, k in enumerate(order)
           if prev is not None and prev[k] != slab[k]]
    return dict(order=order, begin=begin, end=end, halo=halo, kw=kw, mig=mig, slab=slab, nc=nc)


def test_structure_vs_brute_force():
    n = 300
    pts = W.random_box(n, (1.0, 0.6, 0.5), seed=7).astype(np.float32)
    # scramble presentation order; ids are not the presentation index
    perm = np.argsort(W.u01(99, np.arange(n), 0))
    pts, ids = pts[perm], perm.astype(np.int64)
    dom_min, dom_max, h = (0.0, 0.0, 0.0), (1.0, 0.6, 0.5), 0.05
    nc = OA.grid_dims(dom_min, dom_max, h)
    assert nc[0] == 10 and nc[2] == 5   # fp32(0.6)/(2 fp32(0.05)) is a hair above 6 -> ncy = 7
    planes = [0, 3, 5, 10]
    prev = np.clip((pts[:, 0] * 3.2).astype(np.int64), 0, 2)
    A = OA.structure(pts, ids, dom_min, dom_max, h, planes, prev)
    Bf = _brute_structure(pts, list(ids), dom_min, dom_max, h, planes, list(prev))
    assert list(A["order"]) == Bf["order"]
    assert list(A["cell_begin"]) == Bf["begin"]
    assert list(A["cell_end"]) == Bf["end"]
    assert [int(x) for x in A["keyword_sorted"]] == Bf["kw"]
    for s in range(3):
        assert list(A["id_sorted"][A["halo"][s][0]]) == Bf["halo"][s][0]
        assert list(A["id_sorted"][A["halo"][s][1]]) == Bf["halo"][s][1]
    assert [tuple(int(x) for x in row) for row in A["migrants"]] == Bf["mig"]
    # invariants
    assert sorted(A["id_sorted"]) == list(range(n))
    assert A["cell_begin"][-1] == n and (np.diff(A["cell_begin"].astype(np.int64)) >= 0).all()
    assert (A["cell_end"][:-1] == A["cell_begin"][1:]).all()
    assert A["owned"].sum() == n
    assert (A["slab_begin"] == np.concatenate([[0], np.cumsum(A["owned"])])).all()
    # migration bookkeeping: what leaves s towards the right enters some s' > s
    m = A["migrants"]
    for s in range(3):
        assert A["mig_count"][s, 0] == np.count_nonzero((m[:, 2] == s) & (m[:, 3] < s))
        assert A["mig_count"][s, 1] == np.count_nonzero((m[:, 2] == s) & (m[:, 3] > s))
    assert A["mig_count"].sum() == len(m) > 0


def test_migration_labels_both_directions_by_hand():
    """"particles are labeled as '1' if they migrated to left, '2' if they migrated to right,
    and '0' if they stayed"; L240: the same 1 / 2 / 0 for left edge / right edge / interior.  Six particles
    on a 6 x 1 x 1 grid (cell side 2h = 1, x = cell + 0.5 exactly), planes 0|2|4|6, previous owners chosen
    so that two moved left, two moved right and two stayed.  Every expected value below is written by
    hand from those two sentences and the keyword layout of include/sph_b200.h (cell in bits 0..27, edge
    label in bits 28..29, migration label in bits 30..31)."""
    pos = np.array([[k + 0.5, 0.5, 0.5] for k in range(6)], dtype=np.float32)
    planes = [0, 2, 4, 6]
    #                 id: 0  1  2  3  4  5        owner now: 0 0 1 1 2 2
    prev = np.array([1, 0, 2, 0, 1, 2], dtype=np.uint8)   # 0: 1->0 left, 2: 2->1 left, 3: 0->1 right, 4: 1->2 right
    slab = np.array([0, 0, 1, 1, 2, 2])
    assert list(OA.mig_label(slab, prev)) == [1, 0, 1, 2, 2, 0]
    assert list(OA.mig_label(slab, None)) == [0] * 6
    assert list(OA.halo_label(np.arange(6), planes)) == [0, 2, 1, 2, 1, 0]
    A = OA.structure(pos, np.arange(6), (0.0, 0.0, 0.0), (6.0, 1.0, 1.0), 0.5, planes, prev)
    assert tuple(A["nc"]) == (6, 1, 1)
    assert [int(k) for k in A["keyword_sorted"]] == [0x40000000, 0x20000001, 0x50000002, 0xA0000003,
                                                     0x90000004, 0x00000005]
    assert [tuple(int(x) for x in row) for row in A["migrants"]] == [(0, 0, 1, 0), (2, 2, 2, 1), (3, 3, 0, 1),
                                                                     (4, 4, 1, 2)]
    # mig_count[s] = (left slab s towards the left, towards the right): 3 left slab 0 rightwards; 0 and 4
    # left slab 1 (one each way); 2 left slab 2 leftwards
    assert A["mig_count"].tolist() == [[0, 1], [1, 1], [1, 0]]


def test_halo_sufficiency_against_brute_force_neighbours():
    """Every neighbour (0 < r < 2h) of a particle owned by slab s is owned by s or is in
    the halo L_s u R_s (halo width = interaction range 2h)."""
    n = 1500
    box = (1.0, 0.5, 0.5)
    pts64 = W.random_box(n, box, seed=3)
    pts = pts64.astype(np.float32)
    h = 0.04
    dom_min, dom_max = (0.0, 0.0, 0.0), box
    nc = OA.grid_dims(dom_min, dom_max, h)
    planes = W.slab_planes(nc[0], 4)
    A = OA.structure(pts, np.arange(n), dom_min, dom_max, h, planes)
    p = OB.make_params(h=float(np.float32(h)))
    pairs = OB.neighbour_pairs(p, pts.astype(np.float64))
    assert len(pairs) > 1000
    slab_by_id = np.empty(n, dtype=np.int64)
    slab_by_id[A["id_sorted"]] = A["slab_sorted"]
    halo_sets = [set(A["id_sorted"][L]) | set(A["id_sorted"][R]) for (L, R) in A["halo"]]
    cross = 0
    for i, j in pairs:
        s = slab_by_id[i]
        if slab_by_id[j] != s:
            cross += 1
            assert j in halo_sets[s]
    assert cross > 0


def test_halo_fraction_eq14():
    """Eq. (14): n_halo/n_sub ~ N 2h / W.  Uniform cube, S slabs of width W/S: one halo
    plane holds ~ n/ncx particles (Poisson), i.e. n_halo/n_sub = S/ncx per side."""
    w = W.uniform_cube(1 << 16)
    nc = OA.grid_dims(w.params["dom_min"], w.params["dom_max"], w.params["h"])
    planes = W.slab_planes(nc[0], w.n_slabs)
    A = OA.structure(w.pos, np.arange(w.n), w.params["dom_min"], w.params["dom_max"],
                     w.params["h"], planes, w.prev_slab)
    expect = w.n / nc[0]
    for s, (L, R) in enumerate(A["halo"]):
        for side, H in (("L", L), ("R", R)):
            if (s == 0 and side == "L") or (s == w.n_slabs - 1 and side == "R"):
                assert len(H) == 0
            else:
                assert abs(len(H) - expect) < 6 * math.sqrt(expect)
    # a few per cent of synthetic migrants
    assert 0 < len(A["migrants"]) < 0.2 * w.n


def test_first_call_has_no_migrants_and_single_slab_no_edges():
    w = W.dam_break(16)
    nc = OA.grid_dims(w.params["dom_min"], w.params["dom_max"], w.params["h"])
    A = OA.structure(w.pos, np.arange(w.n), w.params["dom_min"], w.params["dom_max"],
                     w.params["h"], [0, nc[0]])
    assert len(A["migrants"]) == 0
    assert (A["keyword_sorted"] >> 28 == 0).all()
    assert A["halo"][0][0].size == 0 and A["halo"][0][1].size == 0
    # lattice sanity: 2h = 3dp, so an interior fluid cell holds 27 particles
    occ = np.diff(A["cell_begin"].astype(np.int64))
    assert occ.max() == 27


# ---------------------------------------------------------------- movable slab planes (NEXT-4)
def test_balance_planes_uniform_counts_give_even_planes():
    """Equal counts per plane: the balanced planes are the evenly spaced ones."""
    assert OA.balance_planes([5] * 24, 4) == [0, 6, 12, 18, 24]
    assert OA.balance_planes([1] * 16, 8) == [0, 2, 4, 6, 8, 10, 12, 14, 16]
    assert OA.balance_planes([7] * 9, 1) == [0, 9]


def test_balance_planes_hand_cases():
    # all particles in the first two planes: planes are pushed right only as far as ">= 2 planes
    # per slab" forces them; ties (empty planes all cost the same) go to the LOWEST plane
    assert OA.balance_planes([10, 10, 0, 0, 0, 0, 0, 0], 2) == [0, 2, 8]        # C[2] = 20 > 10: |40 - 20| = 20 at p = 2..6, lowest wins
    # C = 0 1 2 3 103 104 105 106 107; N = 107; S = 2: target 53.5 -> |2C - 107|: p=3: 101, p=4: 99 -> 4
    assert OA.balance_planes([1, 1, 1, 100, 1, 1, 1, 1], 2) == [0, 4, 8]
    # three slabs, dam-break-like: fluid in the left third
    counts = [0, 9, 9, 9, 9, 1, 1, 1, 1, 1, 1, 0]
    pl = OA.balance_planes(counts, 3)
    assert pl == [0, 3, 5, 12]          # N = 42: targets 14, 28; C = 0 0 9 18 27 36 37 ..: |3C - 42| min at p = 3 (12); then |3C - 84| min at p = 5 (24 vs p = 4: 3)
    # ... the second plane: C[4] = 27 -> |81 - 84| = 3 but p must be >= 3 + 2 = 5 -> C[5] = 36 -> 24


def test_balance_planes_brute_force_is_locally_optimal():
    """Each interior plane, given its left neighbour, is the feasible plane closest to its target
    (pure-python search); planes are feasible; the spread of the owned counts never gets worse than
    with evenly spaced planes on a one-sided distribution."""
    rng_counts = (W.u01(77, np.arange(60), 0) ** 3 * 1000).astype(np.int64)
    for S in (2, 3, 5, 8):
        pl = OA.balance_planes(rng_counts, S)
        assert OA.check_planes(pl, 60)
        C = np.concatenate([[0], np.cumsum(rng_counts)])
        N = int(C[-1])
        for s in range(1, S):
            lo, hi = pl[s - 1] + 2, 60 - 2 * (S - s)
            costs = {p: abs(int(C[p]) * S - s * N) for p in range(lo, hi + 1)}
            m = min(costs.values())
            assert pl[s] == min(p for p, c in costs.items() if c == m)
        owned = np.diff(C[pl])
        even = np.diff(C[W.slab_planes(60, S)])
        assert owned.max() <= even.max()


def test_plane_counts_sum_and_match_structure():
    w = W.dam_break(16)
    P = w.params
    cnt = OA.plane_counts(w.pos, P["dom_min"], P["dom_max"], P["h"])
    assert cnt.sum() == w.n
    nc = OA.grid_dims(P["dom_min"], P["dom_max"], P["h"])
    pl = OA.balance_planes(cnt, 3)
    A = OA.structure(w.pos, np.arange(w.n), P["dom_min"], P["dom_max"], P["h"], pl)
    assert A["owned"].sum() == w.n
    B = OA.structure(w.pos, np.arange(w.n), P["dom_min"], P["dom_max"], P["h"], W.slab_planes(nc[0], 3))
    assert A["owned"].max() < B["owned"].max()          # the fluid sits in the left part of the tank


def test_neighbour_pairs_counts_on_an_integer_lattice():
    """Pin of the brute-force neighbour list: unit lattice, h = 1.5 (2h = 3).  Integer vectors with
    0 < |v|^2 < 9: r3(1..8) = 6 + 12 + 8 + 6 + 24 + 24 + 0 + 12 = 92; another r3(9) = 30 sit exactly AT
    r = 2h and count only when the cut-off is a hair larger (strict inequality)."""
    r = W.lattice_block(9, 9, 9, 1.0)
    centre = (4 * 9 + 4) * 9 + 4
    pairs = OB.neighbour_pairs(OB.make_params(h=1.5), r)
    assert np.count_nonzero(pairs[:, 0] == centre) == 92
    assert np.count_nonzero(pairs[:, 1] == centre) == 92                 # symmetric
    assert len(set(map(tuple, pairs))) == len(pairs) and (pairs[:, 0] != pairs[:, 1]).all()
    pairs = OB.neighbour_pairs(OB.make_params(h=1.5 * (1 + 1e-9)), r)
    assert np.count_nonzero(pairs[:, 0] == centre) == 122
    corner = OB.neighbour_pairs(OB.make_params(h=0.5 * (1 + 1e-9)), r)   # 2h = 1+: face neighbours only
    assert np.count_nonzero(corner[:, 0] == 0) == 3 and np.count_nonzero(corner[:, 0] == centre) == 6
