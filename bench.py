#!/usr/bin/env python
"""bench.py - whole-hot-path throughput of the B200 SPH step (BASELINE.json metric:
Mparticle-steps/s on synthetic 3-D dam breaks, radix-sort Gkeys/s, % of roofline).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 0..3] [--impl reference]
    python bench.py --micro 26            # sort/halo microbenchmark at N = 2^26 (configs[4])

One "step" = one sph_step() = all rows of the hot path (keys+tags, radix sort, payload
permutation, cell table, halo gather, migrant compaction, 27-cell interaction, Verlet) over the
whole particle set.  Default workload: BASELINE config 3 (32 M fluid + 2 M boundary particles,
16 logical x-slabs), the size the roofline bars are judged at; its working set (6.7 GB) is far
larger than the 126 MB L2, so no L2 flush is needed between steps.

N > 1 (torchrun): the path has no inter-GPU exchange (BASELINE north_star drops it), so every
rank steps an independent replica ("replicas only", weak scaling); time = max over ranks.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

CONFIG_NB = {0: 16, 1: 100, 2: 200, 3: 317}
METRIC = "Mparticle-steps/s"
FP32_LANES_PER_SM, NUM_SMS = 128, 148
FLOPS_PER_CANDIDATE, FLOPS_PER_PAIR = 8, 32
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the production interaction kernel, from
# an `ncu --set full` capture of this command (DRAM counters cannot be read inside a timed run): config ->
# (bytes, file under profiles/ that holds the capture).  Configs without a capture report null.
IA_TRAFFIC = {3: (3284194000 + 532750848, "ncu capture profiles/r03_ncu_full_config3.md (dram__bytes_read.sum + dram__bytes_write.sum), "
                  "final build of round 3")}
IA_KERNEL = {0: "interact_mma_kernel", 1: "interact_simple_kernel"}
# algorithmic HBM bytes per particle of the memory-bound stages
# dt_reduce (sph_time_step): acc4 16 + velrho4 16 + mumax 4 + idt 4 B read per particle
BYTES = dict(keys=28.0, sort_per_pass=16.0, gather=116.0, verlet=116.0, migrate=4.0, dt_reduce=40.0)


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx = gpu_index
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.idx), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self) -> dict:
        if self.p is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f:
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2])); power.append(float(c[3]))
            except ValueError:
                continue
            for k, nm in enumerate(names):
                if c[5 + k].lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if not sm:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["no samples"])
        return dict(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons),
                    power_w_max=float(max(power)), samples=len(sm))


def oracle_step_sample(w, max_particles: int):
    """Time the oracles, as they stand, on a bounded spatial sample of the workload: the
    particles with the smallest x (a contiguous piece of the tank, boundary included).
    Returns (particles, seconds, cores, description)."""
    from oracle import physics as OB
    from oracle import structure as OA
    n = min(w.n, max_particles)
    if n < w.n:
        xs = np.partition(w.pos[:, 0], n - 1)[n - 1]
        sel = np.nonzero(w.pos[:, 0] <= xs)[0][:n]
    else:
        sel = np.arange(w.n)
    pos, vel, rho, typ = w.pos[sel], w.vel[sel], w.rho[sel], w.type[sel]
    P = w.params
    p = OB.params_from_workload(P)
    OB.lib()
    s = OB.State(pos, vel, rho, typ)
    nc = OA.grid_dims(P["dom_min"], P["dom_max"], P["h"])
    from paper_1210_1017_b200 import workloads as W
    planes = W.slab_planes(nc[0], w.n_slabs)
    t0 = time.perf_counter()
    OA.structure(pos, np.arange(len(sel)), P["dom_min"], P["dom_max"], P["h"], planes)
    OB.step(p, s, w.dt, verlet_ns=P["verlet_ns"])
    dt = time.perf_counter() - t0
    desc = f"{len(sel)} particles of lowest x of {w.name}, 1 step (structure + rates + Verlet)"
    if n < w.n:
        desc += " - a wall-heavy end of the tank: see mean_neighbours against the whole workload's"
    return len(sel), dt, OB.threads(), desc


def mean_neighbours(pos, h, probes: int = 20000) -> float:
    """Descriptive statistic only (scipy k-d tree, not the oracle): mean number of neighbours with
    0 < r < 2h of `probes` evenly spaced particles of the set."""
    from scipy.spatial import cKDTree
    tree = cKDTree(pos.astype(np.float64))
    sel = np.linspace(0, len(pos) - 1, min(probes, len(pos))).astype(np.int64)
    cnt = tree.query_ball_point(pos[sel].astype(np.float64), 2.0 * h * (1.0 - 1e-12), return_length=True)
    return float(np.mean(cnt) - 1.0)


def oracle_sample_neighbours(w, max_particles: int) -> float:
    n = min(w.n, max_particles)
    if n < w.n:
        xs = np.partition(w.pos[:, 0], n - 1)[n - 1]
        sel = np.nonzero(w.pos[:, 0] <= xs)[0][:n]
        return mean_neighbours(w.pos[sel], w.params["h"])
    return mean_neighbours(w.pos, w.params["h"])


def oracle_structure_sample(w, planes):
    """Oracle A (structure definition: keys, sort, cell table, slab ranges, halos, migrants), as it
    stands, on the whole workload.  Returns seconds."""
    from oracle import structure as OA
    P = w.params
    t0 = time.perf_counter()
    OA.structure(w.pos, np.arange(w.n), P["dom_min"], P["dom_max"], P["h"], planes, prev_slab=w.prev_slab)
    return time.perf_counter() - t0


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on a bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1210_1017_b200 import workloads as W
    nb = CONFIG_NB[args.config]
    w = W.dam_break(nb)
    budget = args.ref_sample
    n_s, _, cores, desc = oracle_step_sample(w, budget)           # warm-up (builds the library)
    for _ in range(max(0, args.warmup - 1)):
        oracle_step_sample(w, budget)
    t = 0.0
    for _ in range(args.steps):
        _, dt, _, _ = oracle_step_sample(w, budget)
        t += dt
    value = n_s * args.steps / t / 1e6
    line = dict(impl="reference", metric=METRIC, value=value, unit="Mparticle-steps/s", n_gpus=args.gpus,
                steps=args.steps, warmup=args.warmup, ms_per_step=1e3 * t / args.steps,
                higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
                config=dict(workload=f"config{args.config}: {w.name}", n_particles=n_s, sampled=True,
                            n_particles_of_workload=w.n, n_slabs=w.n_slabs, sample=desc),
                cpu_baseline=dict(value=value, unit="Mparticle-steps/s", cores=cores, kind="oracle", sample=desc),
                e2e=dict(value=value, unit="Mparticle-steps/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0),
                gpu_launches=0)
    print(json.dumps(line))


def migrate_bytes(n: int, n_mig: int) -> float:
    """Algorithmic bytes of the migrant compaction: the keyword of every slot of a 4096-slot group that
    holds a migrant (groups without one are skipped: their count was taken by the gather kernel) +
    16 B per record written."""
    return min(4.0 * n, 4.0 * 4096 * n_mig) + 16.0 * n_mig


def stage_entry(ms: float, nbytes, hbm_gbs: float, **extra) -> dict:
    """One HBM-bound stage: algorithmic GB/s and fraction of the measured copy peak.  A stage that moved
    less than 8 MB (no or few migrants, tiny halo planes: about 1 us at the copy bandwidth, less than the
    launch latency of its kernels) is launch latency, not a bandwidth: null."""
    d = dict(ms=ms, **extra)
    if nbytes is None:
        return d
    if nbytes < 8e6:
        d.update(algorithmic_gbs=None, frac_of_hbm_peak=None, note="< 8 MB moved: launch latency, not a bandwidth")
        return d
    gbs = nbytes / (ms * 1e-3) / 1e9
    d.update(algorithmic_gbs=gbs, frac_of_hbm_peak=gbs / hbm_gbs)
    return d


def run_micro(args):
    """Sort/halo microbenchmark (configs[4]); prints its own JSON (not the driver's line)."""
    print(json.dumps(micro_measure(args.micro, args.steps, args.warmup,
                                   cpu_baseline=not args.no_cpu_baseline and args.micro <= 26)))


def micro_measure(log2n: int, steps: int, warmup: int, cpu_baseline: bool, device: str = "cuda:0") -> dict:
    """BASELINE.json configs[4] at N = 2^log2n: uniform-random positions, 8 logical x-slabs, synthetic previous
    owners; every iteration restores the random order (untimed) and times sph_sort_and_cells + sph_build_halos
    with the stage timers.  Returns Gkeys/s and the HBM fraction of every stage."""
    import torch
    from paper_1210_1017_b200 import binding as B
    from paper_1210_1017_b200 import workloads as W
    args = argparse.Namespace(steps=steps, warmup=warmup, micro=log2n, no_cpu_baseline=not cpu_baseline)
    n = 1 << args.micro
    w = W.uniform_cube(n)
    pk = peaks()
    sph = B.Sph(w.params, w.pos, w.vel, w.rho, w.type, prev_slab=w.prev_slab, device=device)
    v = sph.sph_get_view()
    planes = W.slab_planes(v.nc[0], 8)
    sph.sph_set_slabs(planes)
    dpos = torch.from_numpy(w.pos).cuda()
    dvel = torch.from_numpy(w.vel).cuda()
    drho = torch.from_numpy(w.rho).cuda()
    dprev = torch.from_numpy(w.prev_slab).cuda()
    reps = args.steps
    acc = {}
    for it in range(args.warmup + reps):
        sph.sph_set_state(dpos, dvel, drho, None, dprev)          # restore random order (untimed)
        sph.sph_profile_enable(it >= args.warmup)
        sph.sph_sort_and_cells()
        sph.sph_build_halos()
        if it >= args.warmup:
            for k, (ms, c) in sph.sph_profile_read().items():
                acc.setdefault(k, []).append(ms)
    T = sph.view_tensors()
    n_halo = int(T["halo_offset"][-1].item())
    n_mig = int(T["mig_total"].item())
    passes = (v.cell_bits + 7) // 8
    med = {k: float(np.median(x)) for k, x in acc.items() if np.sum(x) > 0}
    byts = dict(keys=BYTES["keys"] * n, sort=BYTES["sort_per_pass"] * passes * n, gather=BYTES["gather"] * n,
                cells=None, halo=72.0 * n_halo, migrate=migrate_bytes(n, n_mig))
    out = dict(workload=w.name, n=n, cell_bits=v.cell_bits, passes=passes, n_halo=n_halo, n_migrants=n_mig,
               sort_gkeys_s=n / (med["sort"] * 1e-3) / 1e9,
               sort_with_keys_gkeys_s=n / ((med["sort"] + med["keys"]) * 1e-3) / 1e9,
               hbm_peak_gbs=pk["hbm_gbs"], peak_source=pk["source"],
               stages={k: stage_entry(med[k], byts[k], pk["hbm_gbs"]) for k in med if k in byts})
    ks_b = byts["keys"] + byts["sort"]
    ks_ms = med["keys"] + med["sort"]
    out["stages"]["keys+sort"] = stage_entry(ks_ms, ks_b, pk["hbm_gbs"])
    if not args.no_cpu_baseline and args.micro <= 26:
        # structure cpu_baseline: Oracle A (numpy; lexsort, searchsorted and filters are single-threaded)
        sec = oracle_structure_sample(w, planes)
        out["cpu_baseline"] = dict(value=n / sec / 1e6, unit="Mkeys/s (structure: keys, sort, cell table, halos, "
                                   "migrants)", cores=1, kind="oracle", seconds=sec,
                                   sample=f"all {n} particles of {w.name}, one structure build")
    # the cell table is written by the gather kernel (short gaps) and the gap-fill kernel of the
    # "cells" stage (long runs of empty cells): one combined figure, 4 B written per cell
    gc_ms = med["gather"] + med["cells"]
    gc_b = byts["gather"] + 4.0 * (v.ncells + 1)
    out["stages"]["gather+cells"] = stage_entry(gc_ms, gc_b, pk["hbm_gbs"])
    out["iterations"] = dict(timed=reps, warmup=args.warmup, figure="median over the timed iterations")
    sph.sph_destroy()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=3, choices=[0, 1, 2, 3])
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--micro", type=int, default=0, help="log2 N of the sort/halo microbenchmark")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--e2e-contexts", type=int, default=3, help="contexts pipelined in the end-to-end measurement")
    ap.add_argument("--cpu-sample", type=int, default=1_500_000, help="particles of the cpu_baseline sample")
    ap.add_argument("--ref-sample", type=int, default=300_000, help="particles per step of --impl reference")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--main-micro", type=int, default=26, metavar="LOG2N",
                    help="after the main measurement (config 3, N = 1 only), run the sort/halo microbenchmark at 2^LOG2N "
                         "in the same process and attach it to the JSON line under 'micro' (0 = skip)")
    ap.add_argument("--variant", type=int, default=0)
    ap.add_argument("--kernel", type=int, default=0, choices=[0, 1],
                    help="smoothing kernel: 0 = Wendland C2 (BASELINE configs), 1 = cubic spline (the paper's own, L81)")
    ap.add_argument("--disorder", type=int, default=0, metavar="K",
                    help="time a DISORDERED fluid instead of the rest-state lattice: scrambled start (random "
                         "velocities 0.1 sqrt(gH), densities rho0 (1 + U(0, 1 %%))) stepped K times before warm-up")
    ap.add_argument("--adaptive", action="store_true", help="timed steps use sph_step_adaptive(cfl = 0.2) (variable dt)")
    args = ap.parse_args()
    if args.steps is None:
        args.steps = 10 if (args.impl == "reference" or args.micro) else {0: 200, 1: 200, 2: 200, 3: 100}[args.config]
    args.warmup = max(args.warmup, 3)

    if args.impl == "reference":
        run_reference(args)
        return
    if args.micro:
        run_micro(args)
        return

    import torch
    from paper_1210_1017_b200 import binding as B      # fails loudly without the CUDA library
    from paper_1210_1017_b200 import replicas as R
    from paper_1210_1017_b200 import workloads as W

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    rep = R.init("nccl")
    rank, world, local = rep.rank, rep.world, rep.local_rank
    torch.cuda.set_device(local)
    pk = peaks()

    nb = CONFIG_NB[args.config]
    w = W.dam_break(nb, scrambled=args.disorder > 0)
    if args.kernel:
        w.params = dict(w.params)
        w.params["kernel"] = args.kernel
    sph = B.Sph(w.params, w.pos, w.vel, w.rho, w.type, device=f"cuda:{local}")
    sph.sph_set_option(B.SPH_OPT_INTERACT_VARIANT, args.variant)
    v = sph.sph_get_view()
    planes = W.slab_planes(v.nc[0], w.n_slabs)
    sph.sph_set_slabs(planes)
    n = w.n
    passes = (v.cell_bits + 7) // 8

    def barrier():
        R.barrier(rep)

    # ---- warm-up (preceded by the steps that let a scrambled start disorder the lattice)
    for _ in range(args.disorder):
        sph.sph_step(w.dt)
    for _ in range(args.warmup):
        sph.sph_step(w.dt)
    assert sph.sph_status() == 0
    # pair statistics of the state the timed region starts from (for the flop count)
    sph.sph_sort_and_cells()
    cand, pairs = sph.sph_pair_stats()
    launches0 = sph.sph_launch_count()

    # ---- timed region: exactly K steps, device-timed, stage timers on the same stream
    sampler = ClockSampler(local)
    sph.sph_profile_enable(True)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler.start()
    ev0.record()
    for _ in range(args.steps):
        if args.adaptive:
            sph.sph_step_adaptive(0.2)
        else:
            sph.sph_step(w.dt)
    ev1.record()
    barrier()
    clocks = sampler.stop()
    ms_total = ev0.elapsed_time(ev1)
    stage = sph.sph_profile_read()
    sph.sph_profile_enable(False)
    launches = sph.sph_launch_count() - launches0
    assert sph.sph_status() == 0, "non-finite state during the timed run"
    rate, ms_total = R.aggregate_rate(rep, float(n) * args.steps, ms_total)   # all replicas / slowest rank
    value = rate / 1e6

    # ---- end-to-end through the C ABI with HOST buffers: upload, step, download, every step
    pin = dict(pos=torch.from_numpy(w.pos).pin_memory(), vel=torch.from_numpy(w.vel).pin_memory(),
               rho=torch.from_numpy(w.rho).pin_memory(), typ=torch.from_numpy(w.type).pin_memory())
    outp = dict(pos=torch.empty((n, 3), dtype=torch.float32).pin_memory(),
                vel=torch.empty((n, 3), dtype=torch.float32).pin_memory(),
                rho=torch.empty(n, dtype=torch.float32).pin_memory())

    def e2e_step(ctx, out):
        ctx.sph_set_state(pin["pos"].numpy(), pin["vel"].numpy(), pin["rho"].numpy(), pin["typ"].numpy())
        ctx.sph_step(w.dt)
        ctx.sph_download(acc=False, drho=False, pinned=out)

    # (a) one context: upload, step, download strictly one after the other
    if args.e2e_steps > 0:
        e2e_step(sph, outp)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.e2e_steps):
        e2e_step(sph, outp)
    torch.cuda.synchronize()
    e2e_single_s = R.max_over_ranks(rep, max(time.perf_counter() - t0, 1e-9))
    e2e_single = world * n * args.e2e_steps / e2e_single_s / 1e6
    # (b) several contexts (default 3) on their own streams, one host thread each: the same three calls per step,
    # but one context's PCIe copies overlap the other's kernels (what a user with a queue of
    # independent jobs does).  (a) is the reported end-to-end value; (b) is printed beside it.
    e2e_value, e2e_ctx = e2e_single, 1
    if args.e2e_steps > 0 and args.e2e_contexts > 1:
        import threading
        ctxs, outs = [sph], [outp]
        for _ in range(args.e2e_contexts - 1):
            c2 = B.Sph(w.params, w.pos, w.vel, w.rho, w.type, device=f"cuda:{local}", stream=torch.cuda.Stream())
            c2.sph_set_option(B.SPH_OPT_INTERACT_VARIANT, args.variant)
            c2.sph_set_slabs(planes)
            ctxs.append(c2)
            outs.append({k: torch.empty_like(v).pin_memory() for k, v in outp.items()})

        def worker(k, steps):
            torch.cuda.set_device(local)
            for _ in range(steps):
                e2e_step(ctxs[k], outs[k])

        def run_all(steps):
            th = [threading.Thread(target=worker, args=(k, steps)) for k in range(len(ctxs))]
            for t in th:
                t.start()
            for t in th:
                t.join()
            torch.cuda.synchronize()

        run_all(1)
        barrier()
        t0 = time.perf_counter()
        run_all(args.e2e_steps)
        e2e_s = R.max_over_ranks(rep, max(time.perf_counter() - t0, 1e-9))
        e2e_value = world * n * args.e2e_steps * len(ctxs) / e2e_s / 1e6
        e2e_ctx = len(ctxs)
        for c2 in ctxs[1:]:
            c2.sph_destroy()
    # e2e.value = ONE simulation: upload, step, download strictly one after the other.  The figure of
    # several independent simulations sharing the GPU (copies of one overlap the kernels of another) is
    # printed beside it under its own key.
    e2e = dict(value=e2e_single, unit="Mparticle-steps/s",
               h2d_bytes_per_step=int(n * (12 + 12 + 4 + 1)), d2h_bytes_per_step=int(n * (12 + 12 + 4)),
               steps=args.e2e_steps, contexts=1,
               api="per step: sph_set_state(host) + sph_step + sph_download(host), pinned buffers, one context",
               pipelined=dict(value=e2e_value, contexts=e2e_ctx, steps=args.e2e_steps * e2e_ctx,
                              note=f"{e2e_ctx} independent simulations on separate streams, one host thread each"))

    if rank != 0:
        R.finalize(rep)
        return

    # ---- roofline of the dominant kernel (interaction): plain FP32 ALUs
    ia_ms, ia_n = stage["interact"]
    ia_ms_avg = ia_ms / max(ia_n, 1)
    flops = FLOPS_PER_CANDIDATE * cand + FLOPS_PER_PAIR * pairs
    achieved = flops / (ia_ms_avg * 1e-3) / 1e12
    peak = NUM_SMS * FP32_LANES_PER_SM * 2 * pk["sm_max_mhz"] * 1e6 / 1e12
    sm_mhz = clocks.get("sm_mhz") or pk["sm_max_mhz"]
    # the FP32 peak this box really sustains: register-resident FMA chains, same process (csrc/fma_peak.cu)
    peak_meas = max(sph.sph_fma_peak(0, 8192), sph.sph_fma_peak(1, 8192))
    traffic, traffic_src = IA_TRAFFIC.get(args.config if not (args.disorder or args.adaptive or args.variant or args.kernel) else None, (None, None))
    roofline = dict(bound="alu", kernel=IA_KERNEL.get(args.variant, "?"), achieved=achieved, peak=peak, unit="TFLOP/s",
                    frac=achieved / peak, traffic=traffic, traffic_source=traffic_src,
                    peak_source=f"148 SMs x 128 FP32 lanes x 2 flop x {pk['sm_max_mhz']:.0f} MHz (max clock, {pk['source']})",
                    peak_measured=peak_meas, frac_of_measured_peak=achieved / peak_meas,
                    peak_measured_source="sph_fma_peak: FFMA / FFMA2 chains in registers, best of the two, this run",
                    frac_at_observed_clock=achieved / (peak * sm_mhz / pk["sm_max_mhz"]),
                    algorithmic_flops_per_launch=flops, candidates=cand, pairs=pairs,
                    avg_launch_ms=ia_ms_avg, share_of_step=ia_ms / ms_total)

    T = sph.view_tensors()
    n_halo = int(T["halo_offset"][-1].item()) if w.n_slabs > 1 else 0
    n_mig = int(T["mig_total"].item())
    byts = dict(keys=BYTES["keys"] * n, sort=BYTES["sort_per_pass"] * passes * n, gather=BYTES["gather"] * n,
                cells=None, halo=72.0 * n_halo, migrate=migrate_bytes(n, n_mig),
                verlet=BYTES["verlet"] * n, dt_reduce=BYTES["dt_reduce"] * n)
    stages = {}
    for k, (ms, c) in stage.items():
        if c == 0:
            continue
        stages[k] = stage_entry(ms / c, byts.get(k), pk["hbm_gbs"], share=ms / ms_total)
    if "gather" in stages and "cells" in stages:      # see run_micro: one combined figure for a3 + a4
        gc_ms = stages["gather"]["ms"] + stages["cells"]["ms"]
        gc_b = byts["gather"] + 4.0 * (v.ncells + 1)
        stages["gather+cells"] = stage_entry(gc_ms, gc_b, pk["hbm_gbs"], share=gc_ms * args.steps / ms_total)
    if "keys" in stages and "sort" in stages:
        ks_ms = stages["keys"]["ms"] + stages["sort"]["ms"]
        stages["keys+sort"] = stage_entry(ks_ms, byts["keys"] + byts["sort"], pk["hbm_gbs"],
                                          share=ks_ms * args.steps / ms_total)
    # ---- BASELINE.json configs[4] on the same line: the >= 60 % HBM bars of the sort and compaction kernels
    # are quoted on the random-order microbenchmark, not on the (nearly sorted) simulation state
    micro = None
    if args.main_micro and world == 1 and args.config == 3 and not (args.adaptive or args.disorder or args.variant or args.kernel):
        sph.sph_destroy()
        del sph, T, pin, outp
        torch.cuda.empty_cache()
        try:
            micro = micro_measure(args.main_micro, 5, 3, cpu_baseline=False, device=f"cuda:{local}")
        except Exception as ex:                                  # the main figures stand on their own
            micro = dict(error=f"{type(ex).__name__}: {ex}")
    cpu = None
    if not args.no_cpu_baseline:
        oracle_step_sample(w, 20_000)                         # builds / warms the oracle library
        n_s, dt_s, cores, desc = oracle_step_sample(w, args.cpu_sample)
        cpu = dict(value=n_s / dt_s / 1e6, unit="Mparticle-steps/s", cores=cores, kind="oracle", sample=desc,
                   seconds=dt_s, mean_neighbours_of_sample=oracle_sample_neighbours(w, args.cpu_sample),
                   mean_neighbours_of_workload=pairs / float(n))

    line = dict(
        metric=METRIC, value=value, unit="Mparticle-steps/s", n_gpus=world, steps=args.steps, warmup=args.warmup,
        ms_per_step=ms_total / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f32",
        data="synthetic",
        config=dict(workload=f"config{args.config}: 3-D dam break, {w.n_fluid} fluid + {n - w.n_fluid} boundary "
                             f"particles, {w.n_slabs} logical x-slabs",
                    state=(f"disordered: scrambled start + {args.disorder} steps before warm-up" if args.disorder
                           else "rest-state lattice with seeded jitter (BASELINE configs)"),
                    smoothing_kernel=("cubic spline (PAPER.md L81)" if args.kernel else "Wendland C2 (BASELINE.json)"),
                    n_particles=n, n_slabs=w.n_slabs, cells=int(v.ncells), cell_bits=int(v.cell_bits),
                    radix_passes=passes, dt=("variable, cfl 0.2" if args.adaptive else w.dt), multi_gpu="replicas only",
                    l2="no flush: per-step working set %.1f GB >> 126 MB L2" % (n * 198e-9)
                    if n > 5_000_000 else "working set fits L2 (small config)"),
        clocks=clocks, e2e=e2e, gpu_launches=int(launches), roofline=roofline, cpu_baseline=cpu,
        sort_gkeys_s=n / (stages["sort"]["ms"] * 1e-3) / 1e9 if "sort" in stages else None,
        stages=stages, micro=micro, hbm_peak_gbs=pk["hbm_gbs"], peak_source=pk["source"])
    print(json.dumps(line))
    R.finalize(rep)


if __name__ == "__main__":
    main()
