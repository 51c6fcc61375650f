"""ORACLE A - structure.  TEST INFRASTRUCTURE ONLY: imported by tests/, by
``__graft_entry__.smoke()`` and by ``bench.py``'s cpu_baseline / ``--impl reference``
legs; never by the product path.  Shares no code with the CUDA path.

Plain numpy definition of the integer structures the SPH neighbour search and the
sort-based sub-domain bookkeeping of arXiv 1210.1017 produce (fp32 positions in,
integers out; the CUDA path must match BIT-EXACTLY):

* cell label of a particle (section 3.1: "the domain space is divided into
  cubic cells of the size of the kernel support domain, namely 2h ... assigns to each
  particle a label corresponding to the cell to which it belongs");
* particles ordered by that label with the particle id as tie-break (L140 "radix sort
  ... to order the array holding the particle identification labels, or IDs, according
  to the cell"; stable order demonstrated by the worked example L242-260);
* index of the first (and last) particle of each cell (L140 "an extra array is generated
  with the index of the first particle of each cell", L276 "first and last particle in a
  given region");
* edge ("halo") labels 0/1/2 (L240) and migration labels 0/1/2 (L264) for 1-D slab
  sub-domains whose edge/halo width is 2h = one cell plane (L192);
* the halo of each sub-domain = edge of its neighbours (L192, L213-218) and the list of
  migrating particles (L198-210).

Readings where the paper is silent (DESIGN.md section "Readings"):
cells are linearised x-major / z-fastest; indices are clamped to the grid; slabs are
aligned to cell planes; the first call has no migrants.

Movable planes: ``balance_planes`` (equalise the owned counts, >= 2 planes per slab).

Pins (tests/test_oracle_structure.py): the paper's printed sort example L242-260
(tests/golden/paper_halo_sort_example.txt); hand-placed particles with exactly
representable coordinates; brute-force set definitions; halo sufficiency against
brute-force neighbours; the halo fraction of Eq. (14) L366.
"""
from __future__ import annotations

import math

import numpy as np

TAG_SHIFT = 28  # keyword = (tag << 28) + cell,  tag = halo_label + (mig_label << 2)


def grid_dims(dom_min, dom_max, h):
    """Number of 2h-cells per axis: ceil((max - min) / (2h)), evaluated in fp64 on the
    fp32 parameter values (L140: cells "of the size of the kernel support domain, 2h")."""
    return tuple(
        max(1, int(math.ceil((float(np.float32(dom_max[k])) - float(np.float32(dom_min[k])))
                             / (2.0 * float(np.float32(h))))))
        for k in range(3))


def cell_coords(pos32, dom_min, h, nc):
    """(cx, cy, cz) of every particle.  Each arithmetic step is one separately rounded
    fp32 operation: inv = 1/(2h); t = (r - dom_min) * inv; c = clamp(floor(t), 0, nc-1)."""
    pos32 = np.asarray(pos32, dtype=np.float32)
    assert np.isfinite(pos32).all(), "non-finite position"
    inv = np.float32(1.0) / (np.float32(2.0) * np.float32(h))
    out = []
    for k in range(3):
        d = pos32[:, k] - np.float32(dom_min[k])          # fp32 subtract
        t = d * inv                                        # fp32 multiply
        assert t.dtype == np.float32
        c = np.floor(t).astype(np.int64)
        out.append(np.clip(c, 0, nc[k] - 1))
    return out[0], out[1], out[2]


def cell_index(cx, cy, cz, nc):
    """x-major, z-fastest linear cell label."""
    return (cx * nc[1] + cy) * nc[2] + cz


def slab_of(cx, planes):
    """Slab s with planes[s] <= cx < planes[s+1]."""
    planes = np.asarray(planes, dtype=np.int64)
    return np.searchsorted(planes, cx, side="right") - 1


def check_planes(planes, ncx):
    planes = [int(p) for p in planes]
    ok = planes[0] == 0 and planes[-1] == ncx
    S = len(planes) - 1
    for s in range(S):
        width = planes[s + 1] - planes[s]
        ok = ok and (width >= 2 or (S == 1 and width >= 1))
    return ok


def halo_label(cx, planes):
    """Edge label (L240): 1 = in the left edge of its slab (first cell plane, slab has a
    left neighbour), 2 = in the right edge (last cell plane, slab has a right neighbour)."""
    planes = np.asarray(planes, dtype=np.int64)
    S = planes.size - 1
    s = slab_of(cx, planes)
    lab = np.zeros(cx.shape, dtype=np.int64)
    lab[(cx == planes[s]) & (s > 0)] = 1
    right = (cx == planes[s + 1] - 1) & (s < S - 1)
    lab[right] = 2
    return lab


def mig_label(slab, prev_slab):
    """Migration label (L264): 1 = migrated to the left, 2 = to the right, 0 = stayed."""
    lab = np.zeros(slab.shape, dtype=np.int64)
    if prev_slab is None:
        return lab
    prev = np.asarray(prev_slab, dtype=np.int64)
    lab[slab < prev] = 1
    lab[slab > prev] = 2
    return lab


def keywords(pos32, dom_min, h, nc, planes, prev_slab=None):
    """uint32 keyword of every particle (caller's order) and its cell label."""
    cx, cy, cz = cell_coords(pos32, dom_min, h, nc)
    cell = cell_index(cx, cy, cz, nc)
    assert cell.max(initial=0) < (1 << TAG_SHIFT)
    s = slab_of(cx, planes)
    tag = halo_label(cx, planes) + (mig_label(s, prev_slab) << 2)
    return ((tag << TAG_SHIFT) + cell).astype(np.uint32), cell


def sort_by_label(labels, ids):
    """Order by (label, id) ascending - the order a stable radix sort of the id array by
    label gives when ids start ascending (worked example L242-260)."""
    return np.lexsort((np.asarray(ids), np.asarray(labels)))


def cell_table(sorted_cells, ncells):
    """cellBegin[c] = lower_bound, cellEnd[c] = upper_bound of c in the sorted labels,
    for every c in [0, ncells]; empty cell => begin == end."""
    c = np.arange(ncells + 1, dtype=np.int64)
    begin = np.searchsorted(sorted_cells, c, side="left").astype(np.uint32)
    end = np.searchsorted(sorted_cells, c, side="right").astype(np.uint32)
    return begin, end


def plane_counts(pos32, dom_min, dom_max, h):
    """Number of particles in every cell plane along x (bincount of cx)."""
    nc = grid_dims(dom_min, dom_max, h)
    cx, _, _ = cell_coords(pos32, dom_min, h, nc)
    return np.bincount(cx, minlength=nc[0]).astype(np.int64)


def balance_planes(counts, n_slabs):
    """Movable slab planes ("domain decomposition with load balancing", L389;
    SURVEY 8(f) NEXT-4; reading A22): from the per-plane particle counts choose
    planes[0..S] so that every slab owns about N/S particles.  With C[p] = particles in planes
    < p, plane s (s = 1..S-1, left to right) is the p in [planes[s-1] + 2, ncx - 2 (S - s)]
    that minimises |C[p] S - s N| (exact integers), the lowest p on ties; every slab keeps
    at least two cell planes (edge = one plane on each side, reading A14)."""
    counts = [int(c) for c in counts]
    ncx, S = len(counts), int(n_slabs)
    assert S == 1 or ncx >= 2 * S
    C = [0]
    for c in counts:
        C.append(C[-1] + c)
    N = C[-1]
    planes = [0]
    for s in range(1, S):
        lo, hi = planes[-1] + 2, ncx - 2 * (S - s)
        best, best_cost = None, None
        for p in range(lo, hi + 1):                     # plain argmin, first minimum wins
            cost = abs(C[p] * S - s * N)
            if best is None or cost < best_cost:
                best, best_cost = p, cost
        planes.append(best)
    planes.append(ncx)
    return planes


def structure(pos32, ids, dom_min, dom_max, h, planes, prev_slab=None):
    """Everything the CUDA path's a1-a6 steps must reproduce, from the plain definitions.

    pos32/ids/prev_slab are in the caller's current order.  Returns a dict:
      nc, ncells, keyword_sorted (u32), id_sorted, order (caller index of sorted k),
      cell_begin (ncells+1), cell_end, slab_begin (S+1), owned (S),
      halo (list over slabs of (L_ids, R_ids) in sorted order),
      migrants (m,4) int64 rows (id, sortedIndex, prev_slab, slab), mig_count (S,2).
    """
    ids = np.asarray(ids, dtype=np.int64)
    nc = grid_dims(dom_min, dom_max, h)
    ncells = nc[0] * nc[1] * nc[2]
    planes = np.asarray(planes, dtype=np.int64)
    assert check_planes(planes, nc[0])
    S = planes.size - 1
    kw, cell = keywords(pos32, dom_min, h, nc, planes, prev_slab)
    order = np.lexsort((ids, cell))
    kw_s, cell_s, id_s = kw[order], cell[order], ids[order]
    begin, end = cell_table(cell_s, ncells)
    nyz = nc[1] * nc[2]
    slab_begin = begin[planes * nyz]
    cx_s = cell_s // nyz
    slab_s = slab_of(cx_s, planes)
    owned = np.bincount(slab_s, minlength=S)
    # halos by the set definition (linear filter over the sorted sequence)
    halo = []
    for s in range(S):
        L = np.nonzero(cx_s == planes[s] - 1)[0] if s > 0 else np.zeros(0, dtype=np.int64)
        R = np.nonzero(cx_s == planes[s + 1])[0] if s < S - 1 else np.zeros(0, dtype=np.int64)
        halo.append((L, R))
    # migrants
    if prev_slab is None:
        mig = np.zeros((0, 4), dtype=np.int64)
        mig_count = np.zeros((S, 2), dtype=np.int64)
    else:
        prev_s = np.asarray(prev_slab, dtype=np.int64)[order]
        m = np.nonzero(prev_s != slab_s)[0]
        mig = np.stack([id_s[m], m, prev_s[m], slab_s[m]], axis=1)
        mig_count = np.zeros((S, 2), dtype=np.int64)
        for s in range(S):
            mig_count[s, 0] = np.count_nonzero((prev_s[m] == s) & (slab_s[m] < s))   # left s, went left
            mig_count[s, 1] = np.count_nonzero((prev_s[m] == s) & (slab_s[m] > s))   # left s, went right
    return dict(nc=nc, ncells=ncells, keyword_sorted=kw_s, cell_sorted=cell_s, id_sorted=id_s,
                order=order, cell_begin=begin, cell_end=end, slab_begin=slab_begin,
                owned=owned, halo=halo, migrants=mig, mig_count=mig_count, slab_sorted=slab_s)
