#!/usr/bin/env python
"""bench.py -- GLUPS and HBM roofline of the LPC3D propagation step on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--size L]

One "step" is one lattice time step: the whole hot path (propagate + phase-rotate +
FID reduce) over every site of the lattice.  The workload is
the configuration the north star quotes its target on: the 512^3 lattice of
BASELINE.json configs[4] (monolith statistics, fp64, NMR kernel alone).  One step
moves 7.5 GB of state and parameters, far more than the 126 MB L2, so no L2 flush is
needed between steps.

N > 1 (torchrun): ONE lattice split into x-slabs over the ranks: weak
scaling on N stacked copies of the 512^3 lattice (a (512 N) x 512 x 512 lattice; the 512^3 lattice is periodic, so
the stack is continuous across the seams), each rank generating its own planes only, one boundary-plane exchange
per step (NCCL send/recv, or the sweeps' own stores into the neighbours' ghost planes with --slab-direct) and no
per-step collective; value = all sites x steps / the slowest rank's device time.  --replicas runs N independent
lattices instead (no data-path communication).

--impl reference times the CPU oracle (oracle/) as it stands on the host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import lpc_inputs  # noqa: E402

METRIC = "lattice site updates/sec (GLUPS), 1 step = propagate + phase-rotate + FID reduce over all sites"
UNIT = "GLUPS"
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md


def parse():
    p = argparse.ArgumentParser()
    p.add_argument("--gpus", type=int, default=1)
    p.add_argument("--steps", type=int, default=1000)
    p.add_argument("--warmup", type=int, default=100)
    p.add_argument("--impl", default="ours", choices=["ours", "reference"])
    p.add_argument("--size", type=int, default=512, help="lattice edge L of the L^3 workload")
    p.add_argument("--workload", default="sweep", choices=["sweep", "config0", "particle", "monolith", "supercap", "film"],
                   help="sweep: configs[4] L^3 (default, the headline workload); the others are BASELINE.json configs[0..3] "
                        "at their full sizes (particle 128^3, monolith 256^3 + moment fields, supercap 2048x256x256); "
                        "film: the 100x100x300 film-electrode cell of PAPER.md:236-248")
    p.add_argument("--links", action="store_true",
                   help="per-link mobility factors alpha_ij (PAPER.md:105): 0.25 on links that touch a porous site, 1 in the bulk")
    p.add_argument("--moments", type=int, default=0, choices=[0, 3], help="also propagate the 3 VACF fields")
    p.add_argument("--precision", type=int, default=0, choices=[0, 1])
    p.add_argument("--kernel", type=int, default=0, choices=[0, 1, 2, 3])
    p.add_argument("--regions", type=int, default=0, metavar="R",
                   help="label R (1..8) equal x-ranges as regions and record the region-resolved FID G_r[n] as well")
    p.add_argument("--slabs", type=int, default=0, metavar="S",
                   help="run ONE lattice cut into x-slabs, S per rank (SURVEY 8(e)): a plane exchange after every step.  Default: 0 on "
                        "one GPU (the unsplit lattice), 1 with --gpus N > 1")
    p.add_argument("--replicas", action="store_true", help="with --gpus N > 1: N independent lattices instead of one split lattice")
    p.add_argument("--strong", action="store_true",
                   help="with slabs: split the workload's own lattice over the ranks (strong scaling) instead of stacking one copy "
                        "per rank along x (weak scaling, the default)")
    p.add_argument("--slab-direct", action="store_true",
                   help="with --slabs: let the sweeps store their outermost planes into the neighbours' ghost planes themselves "
                        "(lpc_set_halo_peers; other ranks' workspaces are mapped through CUDA IPC) instead of copying / sending them "
                        "after the sweep")
    p.add_argument("--sustained-s", type=float, default=2.0,
                   help="after the K timed steps, time a further block of about this many seconds (at least 200 steps) with its own "
                        "clock record: the rate under the board's power cap (0 = skip)")
    p.add_argument("--time-block", type=int, default=0, choices=[0, 1, 2],
                   help="LPC_OPT_TIME_BLOCK: 0 auto (one step per sweep: measured faster on B200), 1 one step per sweep, 2 two steps per sweep where the lattice allows it")
    p.add_argument("--x-chunk", type=int, default=0, help="LPC_OPT_X_CHUNK: planes per x chunk of the one-step sweeps (0: the library's choice)")
    p.add_argument("--serial-launch", action="store_true", help="LPC_OPT_SERIAL_LAUNCH = 1: plain launches (no programmatic dependent launch)")
    p.add_argument("--full-phase", action="store_true",
                   help="LPC_OPT_FULL_PHASE = 1: the sweeps read cos and sin even where every phase angle is small (default: sin alone)")
    p.add_argument("--print-csrc-hash", action="store_true", help="print the hash profiles/traffic.csv is stamped with and exit")
    p.add_argument("--no-cpu-baseline", action="store_true")
    p.add_argument("--no-e2e", action="store_true")
    p.add_argument("--ref-sample-size", type=int, default=int(os.environ.get("LPC_REF_SAMPLE_L", "256")),
                   help="edge of the sub-lattice the CPU oracle is timed on (cpu_baseline and --impl reference)")
    return p.parse_args()


def load_oracle():
    import importlib.util

    spec = importlib.util.spec_from_file_location("lpc_oracle", os.path.join(ROOT, "oracle", "lpc_oracle.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def workload_name(L, moments, precision, workload="sweep"):
    tail = f"{'fp32' if precision else 'fp64'}, {'NMR + 3 moment fields' if moments else 'NMR kernel alone'}"
    if workload == "sweep":
        return f"configs[4] sweep: {L}^3 periodic, monolith statistics (Gaussian pore field ell=8, 20% blocked), {tail}"
    return {"config0": "configs[0]: 32^3 periodic, 30% blocked iid, dF ~ U[-3,0] kT, delta ~ U[-10,0] ppm",
            "particle": "configs[1] single porous carbon particle: 128^3 periodic, sphere R=48 porous (ell=4, 10% blocked), bulk outside",
            "monolith": "configs[2] carbon monolith: 256^3 periodic, pore field ell=8, 20% blocked",
            "supercap": "configs[3] supercapacitor cell: 2048x256x256, reflective x, two film electrodes + bulk",
            "film": "film-electrode cell (PAPER.md:236-248): 100x100x300, reflective z, particles R=9 at 38% of the electrode volume, "
                    "alpha=0.025"}[workload] + ", " + tail


def make_workload(args):
    """The seeded synthetic lattice of the chosen workload (lpc_inputs) and its moment-field count."""
    if args.workload == "sweep":
        return lpc_inputs.sweep(args.size, n_moments=args.moments)
    if args.workload == "config0":
        return lpc_inputs.config0(n_moments=args.moments)
    if args.workload == "particle":
        return lpc_inputs.particle(n_moments=args.moments)
    if args.workload == "monolith":
        return lpc_inputs.monolith(n_moments=args.moments)
    if args.workload == "film":
        return lpc_inputs.film(n_moments=args.moments)
    return lpc_inputs.supercap(n_moments=args.moments)


def csrc_hash():
    """Hash of the CUDA sources the library is built from.  profiles/traffic.csv carries the hash of the sources its ncu
    captures were taken with; a row with another hash is stale and `roofline.traffic` is reported as null."""
    import hashlib

    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_2603_22553_b200", "csrc")
    for name in sorted(os.listdir(csrc)):
        if name.endswith((".cu", ".cuh")):
            h.update(name.encode())
            h.update(open(os.path.join(csrc, name), "rb").read())
    return h.hexdigest()[:16]


def committed_traffic(key):
    """dram read + write bytes per launch (and launches per step) of the step kernel from the committed `ncu --set full`
    capture: profiles/traffic.csv rows are key,dram_bytes_per_step,csrc_hash,source.  None when missing or stale."""
    tpath = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(tpath):
        return None
    want = csrc_hash()
    for row in open(tpath):
        cols = row.strip().split(",")
        if len(cols) >= 3 and cols[0] == key and cols[2] == want:
            return float(cols[1])
    return None


# --------------------------------------------------------------------------------------------
# CPU oracle timing (cpu_baseline leg and --impl reference)
# --------------------------------------------------------------------------------------------
def _omp_set_threads(n):
    """Thread count of the OpenMP runtime the oracle library uses (the oracle itself is not touched)."""
    import ctypes

    try:
        ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))
        return True
    except OSError:
        return False


def oracle_sample(moments, steps=None, warmup=1, budget_s=12.0, L=256, lat=None, threads=None):
    """Time the oracle on a bounded sample of the workload: an L^3 lattice with the same statistics (or `lat` itself)."""
    orc_mod = load_oracle()
    if lat is None:
        lat = lpc_inputs.sweep(L, n_moments=moments)
    cores_all = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    if threads is not None and not _omp_set_threads(threads):
        return None, 0, 0.0
    try:
        return _oracle_sample(orc_mod, lat, moments, steps, warmup, budget_s, threads if threads is not None else cores_all)
    finally:
        if threads is not None:
            _omp_set_threads(cores_all)


def _oracle_sample(orc_mod, lat, moments, steps, warmup, budget_s, cores):
    L = lat.nx
    cap = 100000
    o = orc_mod.Oracle.from_lattice(lat, n_moments=moments, max_steps=cap)
    o.step(warmup)
    if steps is None:
        t0 = time.perf_counter()
        o.step(1)
        one = time.perf_counter() - t0
        steps = max(2, min(2000, int(budget_s / max(one, 1e-6))))
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    o.close()
    return {
        "value": lat.n_sites * steps / dt / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
        "sample": f"{lat.nx}x{lat.ny}x{lat.nz} lattice with the workload's statistics, {steps} steps after {warmup} warm-up "
                  f"(oracle/lpc_oracle.c, gcc -O2 -fopenmp, {cores} thread(s), {dt:.1f} s)",
    }, steps, dt


def cpu_baseline_record(args, lat):
    """the oracle as it stands on the box's host cores -- OpenMP on all cores on the workload's own
    lattice (>= 3 steps at 512^3), plus the 256^3 sample with all cores and single-threaded.  About 20-30 s in all."""
    full, _, _ = oracle_sample(args.moments, steps=3, warmup=1, lat=lat)
    rec = dict(full)
    small, _, _ = oracle_sample(args.moments, budget_s=6.0, L=args.ref_sample_size)
    rec["sample_256"] = {k: small[k] for k in ("value", "cores", "sample")}
    single, _, _ = oracle_sample(args.moments, budget_s=5.0, L=min(args.ref_sample_size, 128), threads=1)
    if single is not None:
        rec["single_thread"] = {k: single[k] for k in ("value", "cores", "sample")}
    return rec


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cb, steps, dt = oracle_sample(args.moments, steps=args.steps if args.steps <= 200 else None, warmup=max(1, min(args.warmup, 3)),
                                  L=args.ref_sample_size)
    line = {
        "impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": max(1, min(args.warmup, 3)), "ms_per_step": dt / steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args.size, args.moments, 0), "sample": cb["sample"]},
        "cpu_baseline": cb,
        "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))


# --------------------------------------------------------------------------------------------
# clocks
# --------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), [v.strip() for v in line.split(",")]))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        rows = [r for t, r in self.rows if t0 <= t <= t1] or [r for _, r in self.rows]
        sm, mx, reasons, power = [], None, set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0]))
                mx = float(r[1])
            except Exception:
                continue
            try:
                power.append(float(r[2]))
            except Exception:
                pass
            for name, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons), "samples": len(sm),
                "power_w": statistics.median(power) if power else None}


# --------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_2603_22553_b200 as lpc
    from paper_2603_22553_b200 import replicas

    world, rank, local = replicas.env_world()
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"

    L, K, W = args.size, args.steps, args.warmup
    lat = make_workload(args)
    if world > 1 and not args.replicas and not args.slabs:
        args.slabs = 1            # the default multi-GPU run: one lattice, one x-slab per rank
    if args.slabs:
        return run_slabs(args, lat, lpc, world, rank, local, dev)
    n_sites = lat.n_sites
    # pinned host buffers: the inputs of the end-to-end job
    host = [torch.from_numpy(a).pin_memory() for a in (lat.dF, lat.blocked, lat.omega)]
    h2d_job = sum(t.numel() * t.element_size() for t in host)

    sus_cap = 20000 if args.sustained_s > 0 else 0
    sim = lpc.Lattice(lat.shape, bc=lat.bc, precision=args.precision, n_moments=args.moments, dt=lat.dt, a=lat.a,
                      alpha=lat.alpha, max_steps=2 * K + W + 8 + sus_cap, device=dev, link_mobility=1 if args.links else 0,
                      n_regions=args.regions)
    sim.set_kernel(args.kernel)
    if args.time_block:
        sim.set_option(lpc.LPC_OPT_TIME_BLOCK, args.time_block)
    if args.full_phase:
        sim.set_option(lpc.LPC_OPT_FULL_PHASE, 1)
    if args.x_chunk:
        sim.set_option(lpc.LPC_OPT_X_CHUNK, args.x_chunk)
    if args.serial_launch:
        sim.set_option(lpc.LPC_OPT_SERIAL_LAUNCH, 1)
    link = None
    if args.links:
        # reduced mobility under confinement: every link that touches a porous (dF != 0) site
        link = torch.from_numpy(lpc_inputs.confined_links(lat.dF != 0.0, 0.25)).pin_memory()
        h2d_job += link.numel() * link.element_size()

    labels = None
    if args.regions:
        x = np.arange(lat.nx, dtype=np.int64)[:, None, None] * np.ones(lat.shape, dtype=np.int64)
        labels = torch.from_numpy((x * args.regions // lat.nx).astype(np.uint8)).pin_memory()
        h2d_job += labels.numel()

    def set_params():
        sim.set_site_params(*host)
        if link is not None:
            sim.set_link_mobility(link)
        if labels is not None:
            sim.set_regions(labels)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- end-to-end job through the C ABI with host buffers: upload + precompute + K steps, each step's G[n] read back
    e2e = None
    if not args.no_e2e:
        set_params()          # warm the path once (page-in, module load)
        lpc.lpc_step_n(sim.handle, 3)
        barrier()
        t0 = time.perf_counter()
        set_params()
        last = None
        for k in range(K):
            lpc.lpc_step_n(sim.handle, 1)
            last = lpc.lpc_read_fid(sim.handle, k + 1, 1)
        torch.cuda.synchronize()
        t_e2e = time.perf_counter() - t0
        e2e_glups, _ = replicas.aggregate_glups(n_sites * K, t_e2e * 1e3, dev)
        e2e = {"value": e2e_glups, "unit": UNIT,
               "h2d_bytes_per_step": h2d_job / K, "d2h_bytes_per_step": 16,
               "what": "lpc_set_site_params from pinned host arrays (amortised over the K steps) + K x (lpc_step_n(1) + "
                       "lpc_read_fid of that step's sample to the host)"}
        assert np.isfinite(last).all()
    else:
        set_params()

    # ---- device-timed region: W warm-up steps, then exactly K steps between CUDA events on the library's stream
    lpc.lpc_step_n(sim.handle, W)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    l0 = sim.launch_count
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    tw0 = time.perf_counter()
    ev0.record()
    lpc.lpc_step_n(sim.handle, K)
    ev1.record()
    barrier()
    tw1 = time.perf_counter()
    clocks = sampler.stop(tw0, tw1)
    ms = ev0.elapsed_time(ev1)
    launches = sim.launch_count - l0
    value, ms_max = replicas.aggregate_glups(n_sites * K, ms, dev)

    # ---- sustained block: the same loop for about args.sustained_s seconds, its own events and clock record.  The
    # metric is "seconds per time step of propagation" over a long run: under the board's power cap the SM
    # clock settles below the burst clock of a 20-step run.
    sustained = None
    if args.sustained_s > 0:
        n_sus = int(max(200, min(sus_cap, args.sustained_s / max(ms / K * 1e-3, 1e-7))))
        n_sus -= n_sus % 2
        sampler2 = ClockSampler(local)
        sampler2.start()
        time.sleep(0.25)
        es0, es1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        ts0 = time.perf_counter()
        es0.record()
        lpc.lpc_step_n(sim.handle, n_sus)
        es1.record()
        barrier()
        ts1 = time.perf_counter()
        clocks2 = sampler2.stop(ts0, ts1)
        ms_sus = es0.elapsed_time(es1)
        v_sus, ms_sus_max = replicas.aggregate_glups(n_sites * n_sus, ms_sus, dev)
        sustained = {"steps": n_sus, "value": v_sus, "unit": UNIT, "ms_per_step": ms_sus_max / n_sus, "kernel_ms": ms_sus / n_sus,
                     "clocks": clocks2}
    fid = sim.fid()
    assert np.isfinite(fid).all() and abs(fid[0] - 1.0) < (1e-4 if args.precision else 1e-12), "FID series is not sane"

    if rank == 0:
        peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
        if os.path.exists(peaks_path):
            peak, peak_src = float(json.load(open(peaks_path))["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (measured copy)"
        else:
            peak, peak_src = FALLBACK_HBM_GBS, "fallback of B200_PROFILING.md"
        bps = sim.bytes_per_site_step
        # The default workload is one launch of the step kernel per step.  With --moments 3 a step is two sweeps
        # (moment channels, then magnetisation) and the roofline is taken over the pair: algorithmic bytes of
        # the step / time of the step.
        ms_kernel = ms / K                 # this rank's own time per step
        achieved = bps * n_sites / (ms_kernel * 1e-3) / 1e9
        # dram read + write bytes per LAUNCH of the dominant kernel from the committed `ncu --set full` capture of this very
        # source tree (profiles/traffic.csv is stamped with csrc_hash(); a stale row reads as null)
        key = f"{L}^3/m{args.moments}/p{args.precision}" if args.workload == "sweep" else f"{args.workload}/m{args.moments}/p{args.precision}"
        if args.links:
            key += "/links"
        if args.regions:
            key += "/regions"
        if args.time_block == 2:
            key += "/tb2"
        if args.full_phase:
            key += "/fullphase"
        traffic = committed_traffic(key)
        steps_per_launch = K / max(launches, 1)
        # the same step with cos AND sin read (the round-1 layout, SURVEY 8(d)'s "stored phase" row: 56 B in fp64): the rate
        # this run would need on those bytes, i.e. what the byte diet of DESIGN.md section 5 is worth
        sim.set_option(lpc.LPC_OPT_FULL_PHASE, 1)
        bps_cs = sim.bytes_per_site_step
        sim.set_option(lpc.LPC_OPT_FULL_PHASE, 1 if args.full_phase else 0)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if args.precision else "f64", "data": "synthetic",
            "config": {"workload": workload_name(L, args.moments, args.precision, args.workload), "lattice": list(lat.shape),
                       "sites": n_sites, "parallelism": f"{world} independent replica(s), no collective",
                       "l2": (f"working set {bps * n_sites / 1e9:.2f} GB per step >> 126 MB L2, no flush needed"
                              if bps * n_sites > 4 * 126e6 else "working set is L2-sized: not an HBM measurement"),
                       "kernel": {0: "auto", 1: "direct", 2: "tma", 3: "persistent"}[args.kernel],
                       "links": "alpha_ij = 0.25 on links that touch a porous site" if args.links else "none",
                       "regions": args.regions},
            "clocks": clocks,
            "e2e": e2e,
            "gpu_launches": int(launches),
            # achieved = algorithmic bytes of the one-step-per-sweep layout (lpc_bytes_per_site_step: 48 B per site update in
            # fp64 where the sweep reads sin alone) x site updates per launch / launch duration.  With two
            # time steps per sweep a launch updates every site twice, so this EFFECTIVE rate can exceed the HBM peak; `dram_gbs`
            # is what actually crossed HBM (ncu traffic / launch time).
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": traffic, "peak_source": peak_src, "bytes_per_site_step": bps,
                         "kernel_ms": ms_kernel * steps_per_launch, "launches_per_step": launches / K,
                         "time_steps_per_launch": steps_per_launch,
                         "dram_gbs": (traffic / (ms_kernel * steps_per_launch * 1e-3) / 1e9) if traffic else None,
                         "frac_of_8TBs_spec": achieved / 8000.0,
                         "bytes_per_site_step_cos_and_sin": bps_cs, "frac_on_cos_and_sin_bytes": achieved * bps_cs / bps / peak},
        }
        if sustained is not None:
            a_sus = bps * n_sites / (sustained["kernel_ms"] * 1e-3) / 1e9
            sustained["roofline"] = {"achieved": a_sus, "frac": a_sus / peak, "frac_of_8TBs_spec": a_sus / 8000.0}
            line["sustained"] = sustained
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline_record(args, lat) if args.workload == "sweep" else oracle_sample(args.moments, L=args.ref_sample_size)[0]
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def run_slabs(args, lat, lpc, world, rank, local, dev):
    """One lattice over all ranks as x-slabs: per step one sweep per slab and the exchange of the boundary planes
    (device copies inside a process, NCCL send/recv between ranks).  value = sites x steps / slowest rank's time."""
    import torch
    import torch.distributed as dist

    from paper_2603_22553_b200 import slab

    K, W = args.steps, args.warmup

    def factory(shape, bc, **cfg):
        m = lpc.Lattice(shape, bc=bc, device=dev, **cfg)
        m.set_kernel(args.kernel)
        return m

    # weak scaling (default): the global lattice is `world` copies of the workload's lattice stacked along x, and every rank
    # hands in its own copy only (local=True); that needs a lattice that continues into itself (periodic x).  Strong scaling
    # (--strong, or a lattice with walls in x): the workload's own lattice is cut over the ranks.
    weak = (not args.strong) and lat.bc[0] == 0
    gshape = (lat.nx * world, lat.ny, lat.nz) if weak else lat.shape
    ss = slab.SlabSet(gshape, bc=lat.bc, slabs_per_rank=args.slabs, lattice_factory=factory, precision=args.precision,
                      n_moments=args.moments, dt=lat.dt, a=lat.a, alpha=lat.alpha, max_steps=K + W + 8)
    ss.set_site_params(lat.dF, lat.blocked, lat.omega, local=weak)
    n_global = gshape[0] * gshape[1] * gshape[2]
    n_direct = ss.enable_direct_stores(remote=world > 1) if args.slab_direct else 0
    ss.step(W)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    l0 = sum(m.launch_count for m in ss.lat.values())
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    tw0 = time.perf_counter()
    ev0.record()
    ss.step(K)
    ev1.record()
    barrier()
    tw1 = time.perf_counter()
    clocks = sampler.stop(tw0, tw1)
    ms = ev0.elapsed_time(ev1)
    t = torch.tensor([ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_max = float(t.item())
    launches = sum(m.launch_count for m in ss.lat.values()) - l0
    fid = ss.fid()
    assert np.isfinite(fid).all() and abs(fid[0] - 1.0) < (1e-4 if args.precision else 1e-12), "FID series is not sane"
    backend = dist.get_backend() if world > 1 else "none"
    if rank == 0:
        peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
        peak = float(json.load(open(peaks_path))["hbm_gbs"]) if os.path.exists(peaks_path) else FALLBACK_HBM_GBS
        m0 = next(iter(ss.lat.values()))
        bps = m0.bytes_per_site_step
        own = sum(hi - lo for s, (lo, hi) in ss.ranges.items() if s in ss.lat) * lat.ny * lat.nz
        achieved = bps * own / (ms / K * 1e-3) / 1e9      # this rank's sites over this rank's time
        plane_bytes = m0.halo_planes(lpc.LPC_HALO_STATE, 0, lpc.LPC_HALO_SEND).shape[1] * (4 if args.precision else 8)
        n_faces = len(slab.messages(ss.n_slabs, ss.periodic))
        print(json.dumps({
            "metric": METRIC, "value": n_global * K / (ms_max * 1e-3) / 1e9, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak" if weak else "strong", "vs_baseline": None,
            "dtype": "f32" if args.precision else "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.size, args.moments, args.precision, args.workload)
                                   + (f", {world} copies stacked along x" if weak and world > 1 else ""),
                       "lattice": list(gshape), "sites": n_global,
                       "parallelism": f"x-slabs: {ss.n_slabs} slabs over {world} rank(s) (backend {backend}), one plane exchange per step "
                                      f"({2 + args.moments} channel planes of {plane_bytes} B per face, {n_faces} faces); "
                                      f"{n_direct} of this rank's faces stored by the sweeps themselves, the rest copied / sent; no per-step collective",
                       "exchange_bytes_per_step": n_faces * (2 + args.moments) * plane_bytes,
                       "l2": "per-rank working set >> 126 MB L2" if bps * own > 4 * 126e6 else "per-rank working set is L2-sized"},
            "clocks": clocks, "e2e": None, "gpu_launches": int(launches),
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None,
                         "bytes_per_site_step": bps, "kernel_ms": ms / K, "launches_per_step": launches / K},
        }))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    args = parse()
    if args.print_csrc_hash:
        print(csrc_hash())
        return
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
