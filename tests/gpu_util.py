"""Helpers of the -m gpu parity tests: run the CUDA path through the C ABI and compare it with
the oracles element by element."""
import numpy as np

from oracle import physics as OB
from oracle import structure as OA


def u32(t):
    """torch int32 device tensor -> numpy uint32."""
    return t.detach().cpu().numpy().view(np.uint32)


def make_sph(w, max_slabs=16, with_prev=True):
    from paper_1210_1017_b200 import binding as B
    return B.Sph(w.params, w.pos, w.vel, w.rho, w.type,
                 prev_slab=w.prev_slab if with_prev else None, max_slabs=max_slabs)


def compare_structure(sph, w, planes, prev_slab, check_payload=True, check_halos=True, check_halo_payload=None):
    """Bit-exact comparison of everything a1-a6 produce with ORACLE A on the generator's
    inputs.  Returns the oracle dict.  check_payload: the sorted state arrays carry w's bits;
    check_halo_payload (default = check_payload): the halo buffers carry w's bits (they are copies
    made BEFORE the Verlet update, so after sph_step they still hold the pre-step state)."""
    if check_halo_payload is None:
        check_halo_payload = check_payload
    P = w.params
    A = OA.structure(w.pos, np.arange(w.n), P["dom_min"], P["dom_max"], P["h"], planes, prev_slab)
    T = sph.view_tensors()
    v = T["view"]
    assert tuple(v.nc) == tuple(A["nc"]) and v.ncells == A["ncells"]
    assert sph.sph_status() == 0
    kw = u32(T["keyword"])
    idt = u32(T["idt"])
    ids = idt & 0x0FFFFFFF
    assert np.array_equal(kw, A["keyword_sorted"]), "sorted keywords differ"
    assert np.array_equal(ids, A["id_sorted"].astype(np.uint32)), "permutation differs"
    assert np.array_equal((idt >> 31).astype(np.uint8), w.type[A["id_sorted"]])
    assert np.array_equal(u32(T["cell_begin"]), A["cell_begin"]), "cell table differs"
    assert np.array_equal(u32(T["slab_begin"]), A["slab_begin"]), "slab ranges differ"
    if check_payload:
        pos4 = T["pos4"].cpu().numpy()
        vr = T["velrho4"].cpu().numpy()
        o = A["id_sorted"]
        assert np.array_equal(pos4[:, :3].view(np.uint32), w.pos[o].view(np.uint32))
        assert np.array_equal(vr[:, :3].view(np.uint32), w.vel[o].view(np.uint32))
        assert np.array_equal(vr[:, 3].view(np.uint32), w.rho[o].view(np.uint32))
    if check_halos:
        S = len(planes) - 1
        off = u32(T["halo_offset"]).astype(np.int64)
        hid = u32(T["halo_idt"]) & 0x0FFFFFFF
        hpos = T["halo_pos4"].cpu().numpy()
        hvr = T["halo_velrho4"].cpu().numpy()
        for s in range(S):
            for side in (0, 1):
                k = 2 * s + side
                exp = A["id_sorted"][A["halo"][s][side]]
                got = hid[off[k]:off[k + 1]]
                assert np.array_equal(got, exp.astype(np.uint32)), f"halo {s}/{side} membership differs"
                if check_halo_payload and len(exp):
                    assert np.array_equal(hpos[off[k]:off[k + 1], :3].view(np.uint32), w.pos[exp].view(np.uint32))
                    assert np.array_equal(hvr[off[k]:off[k + 1], :3].view(np.uint32), w.vel[exp].view(np.uint32))
        mig = u32(T["migrants"]).astype(np.int64).reshape(-1, 4)
        assert int(u32(T["mig_total"])[0]) == len(A["migrants"])
        assert np.array_equal(mig, A["migrants"]), "migrant records differ"
        assert np.array_equal(u32(T["mig_count"]).astype(np.int64).reshape(S, 2), A["mig_count"])
    return A


def owners_by_id(A, n):
    """Owner slab of every particle id from an ORACLE A result."""
    own = np.empty(n, dtype=np.uint8)
    own[A["id_sorted"]] = A["slab_sorted"].astype(np.uint8)
    return own


def sampled_rate_errors(w, out, ids):
    """Rates of the sampled particle ids against ORACLE B, which evaluates each sampled neighbourhood
    (all particles within 2h per axis) by brute force.  Returns (worst_a, scale_a, worst_d, scale_d)."""
    p = OB.params_from_workload(w.params)
    two_h = 2.0 * w.params["h"]
    worst_a = worst_d = scale_a = scale_d = 0.0
    order = np.argsort(w.pos[:, 0], kind="stable")
    xs = w.pos[order, 0]
    for i in ids:
        pi = w.pos[i].astype(np.float64)
        lo = np.searchsorted(xs, np.float32(pi[0] - two_h * 1.01), side="left")
        hi = np.searchsorted(xs, np.float32(pi[0] + two_h * 1.01), side="right")
        cand = order[lo:hi]
        sub = w.pos[cand].astype(np.float64)
        near = np.sort(cand[(np.abs(sub - pi) <= two_h * 1.001).all(axis=1)])
        k = int(np.nonzero(near == i)[0][0])
        a, d = OB.rates(p, w.pos[near], w.vel[near], w.rho[near], w.type[near], mode=0)
        if w.type[i] == 0:
            worst_a = max(worst_a, np.abs(out["acc"][i] - a[k]).max())
            scale_a = max(scale_a, np.abs(a[k]).max())
        worst_d = max(worst_d, abs(out["drho"][i] - d[k]))
        scale_d = max(scale_d, abs(d[k]))
    return worst_a, scale_a, worst_d, scale_d


def oracle_rates(w, kernel=None, mode=1):
    P = dict(w.params)
    if kernel is not None:
        P["kernel"] = kernel
    p = OB.params_from_workload(P)
    return OB.rates(p, w.pos, w.vel, w.rho, w.type, mode=mode)


def rate_errors(w, got_acc, got_drho, ref_acc, ref_drho):
    """max|err|/max|ref| for d rho/dt (all particles) and a (fluid only); natural scales when
    the reference vanishes (rest state): rho0 sqrt(g H)/h and |g|."""
    P = w.params
    H = w.notes.get("H", 1.0)
    g = abs(P["g"][2]) or 9.81
    fl = w.type == 0
    s_dr = max(np.abs(ref_drho).max(), 1e-300)
    if np.abs(ref_drho).max() == 0:
        s_dr = P["rho0"] * np.sqrt(g * H) / P["h"]
    s_a = np.abs(ref_acc[fl]).max() if fl.any() else 1.0
    if s_a == 0:
        s_a = g
    e_dr = np.abs(got_drho.astype(np.float64) - ref_drho).max() / s_dr
    e_a = np.abs(got_acc[fl].astype(np.float64) - ref_acc[fl]).max() / s_a if fl.any() else 0.0
    return e_dr, e_a


def rel_l2(got, ref):
    d = np.linalg.norm(got.astype(np.float64) - ref)
    s = np.linalg.norm(ref)
    return d / s if s > 0 else d


def position_rounding_floor(pos0_fluid, n_steps):
    """Expected L2 norm of the rounding noise that fp32 POSITIONS pick up in n_steps Verlet updates:
    r+ = fma(dt^2/2, a, fma(dt, v, r)) rounds twice per step at the magnitude of r, each rounding error
    uniform in +-ulp(r)/2 (variance ulp^2/12).  No fp32-state implementation can follow the fp64 oracle's
    DISPLACEMENT more closely than this; it matters where displacements are small against the
    coordinates (config 3: 10 steps move a particle ~3e-5 m at x ~ 0.5 m, ulp = 6e-8 m).  DESIGN.md 2."""
    ulp = np.spacing(np.abs(np.asarray(pos0_fluid, dtype=np.float32))).astype(np.float64)
    return float(np.sqrt(2.0 * n_steps * np.sum(ulp * ulp) / 12.0))
