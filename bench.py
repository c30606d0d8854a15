#!/usr/bin/env python
"""bench.py -- headline measurement: ns per spin update of a full Swendsen-Wang sweep at L=16384, beta_c, q=2
(BASELINE.json metric; config 3 at beta_c).  --gpus N runs N independent replicas, one per GPU (SURVEY 8(e) "replicas only":
weak scaling, no data-path collective); --bands instead shards ONE lattice into N row bands with one seam all-gather per sweep
(strong scaling); --bands-one-gpu G runs that algorithm band after band on one GPU.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--L 16384] [--beta BETA] [--impl ours|reference]

One JSON line on stdout (rank 0).  A "step" is one pass of the whole hot path -- bond activation, tile-local
labelling, seam merge, flatten + flip -- over one L x L lattice.  Inputs (the spin configuration) are resident in
HBM for `value`; `e2e` goes through sw_sweep_host with pinned HOST buffers, copies inside the timed region.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

PAPER_NS_L16384 = 3.573          # Table I, Tesla M2070, q=2, beta_c, L=16384 (context only)
BYTES_PER_SITE_SWEEP = 14.0      # SURVEY 8(d) model (iii) / DESIGN.md: 1 + 4 + 4 + 4 + 1
BYTES_PER_SITE = {"k_scan": 5.0, "k_seam": 0.0, "k_final": 9.0}   # DESIGN.md per-kernel table
PHASES = ["k_scan", "k_seam", "k_final"]
# bond thresholds floor(p 2^32) of BASELINE.json configs[3], as stored (and pinned) in tests/golden/thresholds.txt -- passed to
# sw_set_threshold as integers: no method arithmetic in the bench
PERC_THRESHOLD = {0.3: 1288490188, 0.5: 2147483648, 0.7: 3006477107}
# ncu counters per launch (dram bytes, warp instructions) are NOT constants of this file: they are read from the tracked
# capture profiles/r03_counters.json, which records the hash of the kernel sources it was taken on; if the sources have
# changed since, the fields are reported as null with the reason (ncu_counters below).
COUNTERS_FILE = os.path.join(ROOT, "profiles", "r03_counters.json")
EQUIL_SWEEPS = 100               # untimed sweeps before the timed region: SURVEY 8(d) "time sweeps 50-200", equilibrium state
N_SMSP = 148 * 4
BYTES_PER_SITE_LABEL = 12.25     # sw_label alone = packed bonds 0.25 + 4 + 4 + 4
BYTES_PER_SITE_CUBIC = 15.0      # cubic_kernels.cuh: spin 1 + bond byte 1 + entry 4 | entry 4 + label 4 + spin 1
BETA_C_CUBIC = 0.2216546         # critical coupling of the 3D Ising model (literature value; chooses the workload only)


def kernel_source_hash() -> str:
    """sha256 over the CUDA sources of the library (the GPU box has no .git: a content hash stands in for the commit)."""
    import glob
    import hashlib
    h = hashlib.sha256()
    for f in sorted(glob.glob(os.path.join(ROOT, "paper_1105_5804_b200", "csrc", "*"))):
        with open(f, "rb") as fh:
            h.update(os.path.basename(f).encode() + b"\0" + fh.read())
    return h.hexdigest()[:16]


def ncu_counters(L: int, beta: float):
    """-> (counters per kernel or None, source string)"""
    try:
        with open(COUNTERS_FILE) as f:
            c = json.load(f)
    except Exception:
        return None, "none: profiles/r03_counters.json absent"
    if c.get("source_sha") != kernel_source_hash():
        return None, "stale: profiles/r03_counters.json was captured on kernel sources %s, this run has %s" % (
            c.get("source_sha"), kernel_source_hash())
    if c.get("L") != L or abs(c.get("beta", -1.0) - beta) > 1e-6:
        return None, "profiles/r03_counters.json is for L=%s beta=%s" % (c.get("L"), c.get("beta"))
    return c["kernels"], "profiles/r03_counters.json (ncu --set full, %s, kernel sources %s)" % (c.get("captured"), c.get("source_sha"))


def beta_c_ising() -> float:
    return 0.5 * math.log(1.0 + math.sqrt(2.0))


def measured_peak_gbs():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s; MEASURED_PEAKS.json absent)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 100 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except ValueError:
                continue
            for name, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def aggregate_over_ranks(local_ms: float, local_units: float, dist=None):
    """Whole-job time = max over ranks, whole-job units = sum over ranks (weak scaling, independent replicas).
    `dist` is torch.distributed (initialised) or None for a single process.  Works on gloo (CPU) and nccl."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return local_ms, local_units
    import torch
    dev = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend() == "nccl" else torch.device("cpu")
    t = torch.tensor([local_ms], dtype=torch.float64, device=dev)
    u = torch.tensor([local_units], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


# ------------------------------------------------------------------------------------------------ reference arm
def reference_sample_L(L: int, steps: int, warmup: int, budget_s: float = 150.0, ns_per_site: float = 160.0) -> int:
    """Largest power-of-two lattice <= L whose (steps+warmup) oracle sweeps fit the time budget."""
    per_step = budget_s / max(1, steps + warmup)
    sites = per_step / (ns_per_site * 1e-9)
    Ls = 64
    while Ls * 2 <= L and (Ls * 2) ** 2 <= sites:
        Ls *= 2
    return Ls


def time_oracle(L: int, beta: float, seed: int, steps: int, warmup: int, spins=None):
    """ns per spin update of the oracle as it stands, one host thread (it is serial, like the paper's CPU code P:322)."""
    import oracle
    T = oracle.threshold(2, beta)
    s = oracle.init_spins(L, 2, seed, 1) if spins is None else spins
    t = 0
    for _ in range(warmup):
        oracle.sweep(L, 2, T, seed, t, s); t += 1
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle.sweep(L, 2, T, seed, t, s); t += 1
    dt = time.perf_counter() - t0
    return dt / steps / (L * L) * 1e9, dt / steps * 1e3


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    Ls = reference_sample_L(args.L, args.steps, args.warmup)
    ns, ms = time_oracle(Ls, args.beta, 1, args.steps, args.warmup)
    sample = ("one serial oracle sweep per step on an L=%d periodic lattice at the same beta from a random start "
              "(%d of the workload's %d sites per step), 1 thread" % (Ls, Ls * Ls, args.L * args.L))
    line = {
        "impl": "reference", "metric": "ns_per_spin_update", "value": ns, "unit": "ns", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "i32", "data": "synthetic",
        "config": {"workload": "2D Ising SW sweep, L=%d periodic, beta=%.10f, q=2" % (args.L, args.beta),
                   "L": args.L, "q": 2, "beta": args.beta, "sampled_L": Ls,
                   "note": "each timed step is one oracle sweep of an L=%d lattice (a bounded sample of the L=%d workload)" % (Ls, args.L)},
        "cpu_baseline": {"value": ns, "unit": "ns", "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": ns, "unit": "ns", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------------------ ablation (S:8f row 4)
def run_ablation(args):
    """python bench.py --ablation: the paper's own labelling pipeline (sw_label_paper: self-labelling + relaxation / sewing) next
    to sw_label on the bond sets of equilibrated critical configurations, L = 1024 .. --L.  One JSON line; not a bench line."""
    import torch
    from paper_1105_5804_b200 import binding
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    rows = []
    L = 1024
    while L <= args.L:
        lat = binding.Lattice(L, 2, args.beta, 1, with_bonds=True)
        lat.init_spins(1)
        lat.sweep(EQUIL_SWEEPS)
        lat.activate()
        ref = torch.empty(L * L, dtype=torch.int32, device="cuda")
        lat.label(None, ref)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(5):
            lat.label(None, ref)
        e1.record()
        torch.cuda.synchronize()
        ours = e0.elapsed_time(e1) / 5
        out = torch.empty(L * L, dtype=torch.int32, device="cuda")
        for B in (8, 16, 32):
            for method in (0, 1):
                st = lat.label_paper(method, B, None, out)
                rows.append({"L": L, "B": B, "consolidation": "relaxation" if method == 0 else "sewing",
                             "labels_equal_sw_label": bool(torch.equal(out, ref)), "sw_label_ms": ours,
                             "ms": st["ms_local"] + st["ms_consolidate"] + st["ms_flatten"],
                             # (the one-thread wrap-around step is this repository's reading of P:213 "in an additional step")
                             "ms_without_wrap": st["ms_local"] + st["ms_consolidate"] + st["ms_flatten"] - st["ms_wrap"], **st})
        lat.close()
        L *= 2
    print(json.dumps({"ablation": "paper pipeline (P:152-258) vs sw_label, bonds of equilibrated configurations at beta=%.7f" % args.beta,
                      "rows": rows}), flush=True)
    return 0


# ------------------------------------------------------------------------------------------------ the other BASELINE.json configs
def per_config_leg(binding, torch, device):
    """ns per spin update of the BASELINE.json configs that are not the headline (north_star: "ns/spin-update reported per
    config"): configs[0] L=64, configs[1] L=1024 cold, configs[3] percolation labelling at p = 0.3 / 0.7, configs[4] q=4 Potts
    L=4096 and Wolff steps on L=4096.  Small lattices are latency bound, not a roofline statement."""
    stream = torch.cuda.current_stream()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def timed(fn, n):
        torch.cuda.synchronize(); ev0.record(stream); fn(n); ev1.record(stream); torch.cuda.synchronize()
        return ev0.elapsed_time(ev1) / n

    out = {}
    for name, L, q, beta, mode, equil, n in (("configs[0] 2D Ising L=64 beta_c", 64, 2, beta_c_ising(), 1, 100, 1000),
                                             ("configs[1] 2D Ising L=1024 beta_c cold start", 1024, 2, beta_c_ising(), 0, 100, 900),
                                             ("configs[4] q=4 Potts L=4096 beta_c=ln 3", 4096, 4, math.log(3.0), 1, 100, 400)):
        lat = binding.Lattice(L, q, beta, 1, device=device)
        lat.init_spins(mode); lat.sweep(equil)
        ms = timed(lat.sweep, n)
        o = lat.observables(clusters=False)
        out[name] = {"ms_per_sweep": ms, "ns_per_spin_update": ms * 1e6 / (L * L), "sweeps": n,
                     "energy_per_site": o["energy"] / (L * L)}
        lat.close()
    L = 4096
    lat = binding.Lattice(L, 2, beta_c_ising(), 1, device=device)
    lat.init_spins(1); lat.sweep(200)
    torch.cuda.synchronize(); ev0.record(stream); sizes = lat.wolff_step(500); ev1.record(stream); torch.cuda.synchronize()
    ms = ev0.elapsed_time(ev1) / 500
    out["configs[4] Wolff steps, 2D Ising L=4096 beta_c (label everything)"] = {
        "ms_per_step": ms, "mean_cluster_sites": sum(sizes) / 500.0, "ns_per_cluster_site": ms * 1e6 / max(1.0, sum(sizes) / 500.0)}
    # the few-cluster variant on the same lattice: 64 seed points, p_flip = 0.7 (threshold as stored
    # for percolation p = 0.7: the same integer floor(0.7 2^32))
    torch.cuda.synchronize(); ev0.record(stream); flipped = lat.fewcluster_step(500, 64, PERC_THRESHOLD[0.7]); ev1.record(stream)
    torch.cuda.synchronize()
    ms = ev0.elapsed_time(ev1) / 500
    out["few-cluster steps (64 seeds, p_flip=0.7), 2D Ising L=4096 beta_c"] = {
        "ms_per_step": ms, "mean_flipped_sites": sum(flipped) / 500.0, "ns_per_flipped_site": ms * 1e6 / max(1.0, sum(flipped) / 500.0)}
    lat.close()
    L = 16384
    latp = binding.Lattice(L, 2, 0.1, 1, device=device, with_bonds=True)
    latp.init_spins(0)
    for pbond in (0.3, 0.7):
        latp.set_threshold(PERC_THRESHOLD[pbond])
        latp.activate(); latp.label()
        ms = timed(lambda n: [latp.label() for _ in range(n)], 10)
        cs = latp.cluster_stats()
        out["configs[3] bond percolation labelling L=16384 p=%.1f" % pbond] = {
            "ms": ms, "ns_per_site": ms * 1e6 / (L * L), "GB/s": BYTES_PER_SITE_LABEL * L * L / (ms * 1e-3) / 1e9,
            "clusters_per_site": cs["n_clusters"] / (L * L), "largest_cluster_fraction": cs["max_cluster"] / (L * L)}
    latp.close()
    return out


# ------------------------------------------------------------------------------------------------ simple cubic lattice
def cubic_leg(binding, torch, device, sizes):
    """SW sweeps of the 3D Ising model at its critical coupling on L^3 periodic lattices: (L, timed sweeps) per entry."""
    stream = torch.cuda.current_stream()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    cubic = {}
    for L3, nsw in sizes:
        N3 = L3 ** 3
        l3 = binding.Lattice(L3, 2, BETA_C_CUBIC, 1, device=device, dim=3)
        l3.init_spins(1)
        l3.sweep(60)
        torch.cuda.synchronize()
        ev0.record(stream)
        l3.sweep(nsw)
        ev1.record(stream)
        torch.cuda.synchronize()
        ms3 = ev0.elapsed_time(ev1) / nsw
        l3.profile_enable(True); l3.sweep(nsw); ph3, n3 = l3.profile_read(); l3.profile_enable(False)
        o3 = l3.observables()
        gbs3 = BYTES_PER_SITE_CUBIC * N3 / (ms3 * 1e-3) / 1e9
        cubic["L%d" % L3] = {"workload": "3D Ising (q=2) SW sweep, %d^3 periodic simple cubic lattice, beta=%.7f, 60 untimed + %d timed sweeps"
                                         % (L3, BETA_C_CUBIC, nsw),
                             "ms_per_step": ms3, "ns_per_spin_update": ms3 * 1e6 / N3,
                             "algorithmic_bytes_per_site": BYTES_PER_SITE_CUBIC, "GB/s": gbs3,
                             "frac_of_measured_peak": gbs3 / measured_peak_gbs()[0],
                             "kernel_ms": {name: ph3[i] / max(1, n3) for i, name in enumerate(["k3_local", "k3_faces", "k3_final"])},
                             "state": {"energy_per_site": o3["energy"] / N3, "magnetisation_per_site": o3["magnetisation"] / N3,
                                       "clusters_per_site": o3["n_clusters"] / N3,
                                       "largest_cluster_fraction": o3["max_cluster"] / N3, "counter": o3["counter"]}}
        l3.close()
    return cubic


def run_cubic_only(args):
    """python bench.py --only-cubic: the simple cubic legs alone (used for the ncu capture of the k3_* kernels)."""
    import torch
    from paper_1105_5804_b200 import binding
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    print(json.dumps({"cubic": cubic_leg(binding, torch, "cuda:0", ((256, 10),))}), flush=True)
    return 0


# ------------------------------------------------------------------------------------------------ row bands (S:8f row 3)
def run_bands(args):
    """python -m torch.distributed.run ... bench.py --gpus N --bands: ONE L x L lattice sharded into N row bands, one per GPU
    (paper_1105_5804_b200/bands.py: a halo row of spins and two rows of roots are all-gathered per sweep).  Strong scaling:
    the work is fixed, value = N sites / time.  Not the default (BASELINE.json: one GPU; `--gpus N` alone runs replicas)."""
    import torch
    import torch.distributed as dist
    from paper_1105_5804_b200 import bands
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world < 2:
        raise SystemExit("--bands needs WORLD_SIZE >= 2 (torchrun); with one GPU run bench.py without it")
    torch.cuda.set_device(local_rank)
    dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    L, beta, N = args.L, args.beta, args.L * args.L
    band = bands.DistBand(L, 2, beta, 1, dist, "cuda:%d" % local_rank)
    band.init_spins(1)
    band.sweep(max(EQUIL_SWEEPS, args.warmup))
    stream = torch.cuda.current_stream()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    dist.barrier(); torch.cuda.synchronize()
    ev0.record(stream)
    band.sweep(args.steps)
    ev1.record(stream)
    dist.barrier(); torch.cuda.synchronize()
    t = torch.tensor([ev0.elapsed_time(ev1)], dtype=torch.float64, device="cuda")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms = float(t.item())
    c = band.counters()
    if rank == 0:
        ms = total_ms / args.steps
        print(json.dumps({
            "metric": "ns_per_spin_update", "value": ms * 1e6 / N, "unit": "ns", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": False, "scaling": "strong", "vs_baseline": None,
            "dtype": "i32", "data": "synthetic",
            "config": {"workload": "2D Ising (q=2) Swendsen-Wang, ONE L=%d periodic lattice in %d row bands, beta=%.10f" % (L, world, beta),
                       "L": L, "q": 2, "beta": beta, "sites_per_step": N, "bands": world,
                       "exchange_bytes_per_rank_and_sweep": L + 8 * L,
                       "equilibration": "%d untimed sweeps" % max(EQUIL_SWEEPS, args.warmup)},
            "state": {"clusters_per_site": c["n_clusters"] / N, "active_bonds_per_site": c["n_active_bonds"] / N,
                      "energy_per_site_before_last_sweep": -(2 * c["sat_before"] - 2 * N) / N},
            "frac_of_8TBps_nominal_per_gpu": BYTES_PER_SITE_SWEEP * N / world / (ms * 1e-3) / 1e9 / 8000.0}), flush=True)
    band.close()
    dist.destroy_process_group()
    return 0


def run_bands_one_gpu(args):
    """python bench.py --bands-one-gpu G: the G-band algorithm run band after band on ONE GPU (bands.BandGroup): what the sharded
    path costs in total GPU work next to sw_sweep (same lattice, same result) -- the per-band share is what one of G GPUs would
    spend, link latency aside.  One JSON line; not a bench line."""
    import torch
    from paper_1105_5804_b200 import bands, binding
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    L, beta, N, G = args.L, args.beta, args.L * args.L, args.bands_one_gpu
    if args.steps < 4:
        raise SystemExit("--bands-one-gpu needs --steps >= 4: three of the group's sweeps are untimed warm-up, the rest are timed")
    n_timed = args.steps - 3
    ref = binding.Lattice(L, 2, beta, 1)
    ref.init_spins(1); ref.sweep(EQUIL_SWEEPS)
    spins = ref.spins.clone(); t0 = ref.get_counter()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize(); ev0.record(); ref.sweep(args.steps); ev1.record(); torch.cuda.synchronize()
    ms_ref = ev0.elapsed_time(ev1) / args.steps
    grp = bands.BandGroup(L, 2, beta, 1, G)
    for lat in grp.lats:                                  # the same equilibrated state on every band
        lat.spins.copy_(spins); lat.set_counter(t0)
    grp.sweep(3)
    torch.cuda.synchronize(); ev0.record(); grp.sweep(n_timed); ev1.record(); torch.cuda.synchronize()
    ms_grp = ev0.elapsed_time(ev1) / n_timed
    same = bool(torch.equal(torch.from_numpy(grp.spins_host()), ref.spins.cpu()))
    print(json.dumps({"bands_one_gpu": G, "L": L, "beta": beta, "sw_sweep_ms": ms_ref, "all_bands_ms": ms_grp,
                      "per_band_ms": ms_grp / G, "work_inflation": ms_grp / ms_ref,
                      "sw_sweep_timed_sweeps": args.steps, "bands_timed_sweeps": n_timed, "bands_warmup_sweeps": 3,
                      "spins_equal_single_gpu_chain_after_%d_sweeps" % args.steps: same}), flush=True)
    grp.close(); ref.close()
    return 0


# ------------------------------------------------------------------------------------------------ our arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1105_5804_b200 import binding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    device = "cuda:%d" % local_rank

    L, beta, N = args.L, args.beta, args.L * args.L
    lat = binding.Lattice(L, 2, beta, 1 + rank, device=device)        # one independent replica per rank
    lat.init_spins(1)
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def state_of(l):
        o = l.observables()
        return {"energy_per_site": o["energy"] / N, "magnetisation_per_site": o["magnetisation"] / N,
                "clusters_per_site": o["n_clusters"] / N, "largest_cluster_fraction": o["max_cluster"] / N,
                "counter": o["counter"]}

    # ---- device-resident timing ----------------------------------------------------------------------------
    # the timed configurations are equilibrium ones whatever --warmup says: at least EQUIL_SWEEPS
    # untimed sweeps from the random start, then the W warm-up sweeps of the contract, then the K timed ones
    lat.sweep(max(0, EQUIL_SWEEPS - args.warmup))
    lat.sweep(args.warmup)
    state_before = state_of(lat) if rank == 0 else None
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    l0 = lat.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record(stream)
    lat.sweep(args.steps)
    ev1.record(stream)
    barrier()
    local_ms = ev0.elapsed_time(ev1)
    launches = lat.launch_count() - l0
    clocks = sampler.stop() if rank == 0 else None
    total_ms, total_units = aggregate_over_ranks(local_ms, float(N) * args.steps, dist if world > 1 else None)
    ms_per_step = total_ms / args.steps
    ns_per_spin = total_ms * 1e6 / total_units

    # ---- per-kernel split (instrumented pass, same state, same stream) ---------------------------------------
    prof_steps = min(args.steps, 64)
    lat.profile_enable(True)
    lat.sweep(prof_steps)
    phase_ms, nprof = lat.profile_read()
    lat.profile_enable(False)
    per_kernel = {name: phase_ms[i] / max(1, nprof) for i, name in enumerate(PHASES)}
    state_after = state_of(lat) if rank == 0 else None

    # ---- labelling alone (BASELINE.json configs[3], metric "labelling GB/s"): bond percolation at p = 1/2 --------------
    labelling = None
    if rank == 0 and not args.no_labelling:
        latp = binding.Lattice(L, 2, beta, 1, device=device, with_bonds=True)
        latp.init_spins(0)                                            # cold spins: every bond is satisfied
        latp.set_threshold(1 << 31)                                   # floor(0.5 * 2^32): each bond open with p = 1/2
        latp.activate()
        for _ in range(3):
            latp.label()
        torch.cuda.synchronize()
        nrep = 20
        ev0.record(stream)
        for _ in range(nrep):
            latp.activate()                                           # materialised packed bonds (a1 alone)
        ev1.record(stream)
        torch.cuda.synchronize()
        act_ms = ev0.elapsed_time(ev1) / nrep
        ev0.record(stream)
        for _ in range(nrep):
            latp.label()
        ev1.record(stream)
        torch.cuda.synchronize()
        lab_ms = ev0.elapsed_time(ev1) / nrep
        latp.profile_enable(True)
        for _ in range(nrep):
            latp.label()
        lab_phase, nlab = latp.profile_read()
        latp.profile_enable(False)
        cs = latp.cluster_stats()
        peak_l, _ = measured_peak_gbs()
        gbs = BYTES_PER_SITE_LABEL * N / (lab_ms * 1e-3) / 1e9
        labelling = {"workload": "sw_label on i.i.d. bonds, p=0.5, L=%d (packed bonds -> canonical int32 labels)" % L,
                     "ms": lab_ms, "ns_per_site": lab_ms * 1e6 / N, "algorithmic_bytes_per_site": BYTES_PER_SITE_LABEL,
                     "GB/s": gbs, "frac_of_measured_peak": gbs / peak_l, "frac_of_8TBps_nominal": gbs / 8000.0,
                     "kernel_ms": {name: lab_phase[i] / max(1, nlab) for i, name in enumerate(PHASES)},
                     "clusters_per_site": cs["n_clusters"] / N,
                     "activation_only": {"what": "sw_activate: spins -> packed bonds (1.25 B/site), not on the sweep path "
                                                 "(a sweep draws its bonds inside k_scan)", "ms": act_ms,
                                         "ns_per_site": act_ms * 1e6 / N}}
        latp.close()

    # ---- the other temperatures of BASELINE.json configs[2] (short runs; the headline stays beta_c) -------------------
    other_betas = None
    if rank == 0 and not args.no_other_betas:
        other_betas = {}
        for b in (0.40, 0.50):
            lb = binding.Lattice(L, 2, b, 1, device=device)
            lb.init_spins(1)
            lb.sweep(EQUIL_SWEEPS)
            torch.cuda.synchronize()
            ev0.record(stream)
            lb.sweep(100)
            ev1.record(stream)
            torch.cuda.synchronize()
            ms = ev0.elapsed_time(ev1) / 100
            lb.profile_enable(True); lb.sweep(50); ph, nb = lb.profile_read(); lb.profile_enable(False)
            other_betas["%.2f" % b] = {"ms_per_step": ms, "ns_per_spin_update": ms * 1e6 / N,
                                       "frac_of_8TBps_nominal": BYTES_PER_SITE_SWEEP * N / (ms * 1e-3) / 1e9 / 8000.0,
                                       "kernel_ms": {name: ph[i] / max(1, nb) for i, name in enumerate(PHASES)},
                                       "state": state_of(lb)}
            lb.close()

    # ---- simple cubic lattice: a second workload, 3D Ising at its critical coupling ------------------
    cubic = cubic_leg(binding, torch, device, ((256, 50), (512, 20))) if rank == 0 and not args.no_cubic else None

    per_config = per_config_leg(binding, torch, device) if rank == 0 and not args.no_per_config else None

    # ---- end to end through the host-buffer entry point ----------------------------------------------------
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    h_in = torch.empty(N, dtype=torch.int8).pin_memory()
    h_out = torch.empty(N, dtype=torch.int8).pin_memory()
    h_in.copy_(lat.spins.cpu())
    lat.sweep_host(h_in, 1, h_out, None, obs_flags=binding.OBS_SPINS)  # warm-up
    barrier()
    ev0.record(stream)
    for _ in range(e2e_steps):
        o = lat.sweep_host(h_in, 1, h_out, None, obs_flags=binding.OBS_SPINS)   # H2D spins, 1 sweep, D2H spins + E, M, counts
        h_in, h_out = h_out, h_in
    ev1.record(stream)
    barrier()
    e2e_ms, e2e_units = aggregate_over_ranks(ev0.elapsed_time(ev1), float(N) * e2e_steps, dist if world > 1 else None)
    e2e_ns = e2e_ms * 1e6 / e2e_units
    # the same call with the 4N bytes of labels copied back as well (rank 0, two steps: a second figure, not the e2e value)
    e2e_labels = None
    if rank == 0 and not args.no_e2e_labels:
        h_lab = torch.empty(N, dtype=torch.int32).pin_memory()
        lat.sweep_host(h_in, 1, h_out, h_lab, obs_flags=binding.OBS_SPINS)
        torch.cuda.synchronize(device)
        ev0.record(stream)
        for _ in range(2):
            lat.sweep_host(h_in, 1, h_out, h_lab, obs_flags=binding.OBS_SPINS)
            h_in, h_out = h_out, h_in
        ev1.record(stream)
        torch.cuda.synchronize(device)
        ms_lab = ev0.elapsed_time(ev1) / 2
        e2e_labels = {"ms_per_step": ms_lab, "ns_per_spin_update": ms_lab * 1e6 / N, "h2d_bytes_per_step": N,
                      "d2h_bytes_per_step": N + 4 * N + 128, "steps": 2,
                      "what": "as e2e, plus the int32 labels of the sweep copied to pinned host memory"}
        del h_lab

    if rank != 0:
        lat.close()
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel ---------------------------------------------------------------------
    peak, peak_src = measured_peak_gbs()
    dom = max(("k_scan", "k_final"), key=lambda k: per_kernel[k])
    dom_bytes = BYTES_PER_SITE[dom] * N
    achieved = dom_bytes / (per_kernel[dom] * 1e-3) / 1e9
    counters, counters_src = ncu_counters(L, beta)
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": counters[dom]["dram_bytes"] if counters else None,
                "traffic_source": counters_src, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": dom_bytes, "kernel_ms": per_kernel[dom],
                "kernel_ms_all": per_kernel,
                "kernel_share_of_step": per_kernel[dom] / max(1e-12, sum(per_kernel.values())),
                "sweep": {"algorithmic_bytes": BYTES_PER_SITE_SWEEP * N,
                          "achieved": BYTES_PER_SITE_SWEEP * N / (ms_per_step * 1e-3) / 1e9,
                          "frac_of_measured_peak": BYTES_PER_SITE_SWEEP * N / (ms_per_step * 1e-3) / 1e9 / peak,
                          "frac_of_8TBps_nominal": BYTES_PER_SITE_SWEEP * N / (ms_per_step * 1e-3) / 1e9 / 8000.0,
                          "frac_compulsory_6B_of_measured_peak": 6.0 * N / (ms_per_step * 1e-3) / 1e9 / peak}}

    if counters and clocks and clocks.get("sm_mhz"):
        # issue-slot view: warp instructions per launch (ncu) / (SM sub-partitions x clock x kernel time); peak 1 per cycle
        roofline["alu"] = {name: {"warp_inst": counters[name]["warp_inst"],
                                  "issue_frac": counters[name]["warp_inst"] / (N_SMSP * clocks["sm_mhz"] * 1e6 * per_kernel[name] * 1e-3)}
                           for name in PHASES}

    # ---- the oracle on this box's host cores, bounded sample ---------------------------------------------------
    cpu = None
    if not args.no_cpu_baseline:
        # the oracle as it stands, one thread, on the workload itself -- 3 sweeps of the L x L lattice from the
        # equilibrated GPU state (about 15 s each at L=16384).  Smaller budgets (--cpu-sweeps 0) fall back to an L=4096 sample.
        import oracle
        T = oracle.threshold(2, beta)
        if args.cpu_sweeps > 0:
            Ls, nsw = L, args.cpu_sweeps
            s = lat.spins_host().copy()
            t_start = lat.get_counter()
        else:
            Ls, nsw = min(L, 4096), 12
            lat_s = binding.Lattice(Ls, 2, beta, 1, device=device)
            lat_s.init_spins(1)
            lat_s.sweep(EQUIL_SWEEPS)
            s = lat_s.spins_host().copy()
            t_start = lat_s.get_counter()
            lat_s.close()
        t0 = time.perf_counter()
        for k in range(nsw):
            oracle.sweep(Ls, 2, T, 1, t_start + k, s)
        dt = time.perf_counter() - t0
        cpu = {"value": dt / nsw / (Ls * Ls) * 1e9, "unit": "ns", "cores": 1, "kind": "oracle",
               "sample": "%d serial oracle sweeps of the L=%d lattice at the same beta, started from the state the GPU "
                         "chain had reached after %d sweeps (%.1f s of CPU work; host has %d cores, the oracle uses 1; "
                         "built %s)" % (nsw, Ls, t_start, dt, os.cpu_count() or 0, oracle.build_flags())}

    line = {
        "metric": "ns_per_spin_update", "value": ns_per_spin, "unit": "ns", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": False, "scaling": "weak",
        "vs_baseline": ns_per_spin / PAPER_NS_L16384 if (L == 16384 and abs(beta - beta_c_ising()) < 1e-9) else None,
        "dtype": "i32", "data": "synthetic",
        "config": {"workload": "BASELINE.json configs[2] at beta_c: 2D Ising (q=2) Swendsen-Wang, L=%d periodic, "
                               "beta=%.10f, random +-1 start from seed, int8 spins / int32 labels" % (L, beta),
                   "L": L, "q": 2, "beta": beta, "sites_per_step": N, "replicas": world,
                   "l2_policy": "inputs larger than L2: spins %d MiB + labels %d MiB per step vs 126 MB L2"
                                % (N >> 20, (4 * N) >> 20),
                   "equilibration": "%d untimed sweeps from the random start before the timed region" % max(EQUIL_SWEEPS, args.warmup),
                   "sweeps_per_s": 1e3 / ms_per_step * world},
        "clocks": clocks,
        "e2e": {"value": e2e_ns, "unit": "ns", "h2d_bytes_per_step": N, "d2h_bytes_per_step": N + 128,
                "steps": e2e_steps, "ms_per_step": e2e_ms / e2e_steps,
                "what": "sw_sweep_host_ex(SW_OBS_SPINS): pinned host spins -> device, one sweep, spins + sw_obs (energy, magnetisation, "
                        "state counts, cluster and bond counts; no cluster-size pass) back to the host; the labels stay on the device",
                "with_labels_copied_back": e2e_labels},
        "gpu_launches": launches,
        "roofline": roofline,
        "cpu_baseline": cpu,
        "labelling": labelling,
        "other_betas": other_betas,
        "cubic": cubic,
        "per_config": per_config,
        "state_before_timed_region": state_before,
        "state": state_after,
    }
    print(json.dumps(line), flush=True)
    lat.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=50)
    ap.add_argument("--L", type=int, default=16384)
    ap.add_argument("--beta", type=float, default=beta_c_ising())
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e-labels", action="store_true", help="skip the second end-to-end figure (labels copied back too; 1 GiB pinned)")
    ap.add_argument("--no-labelling", action="store_true")
    ap.add_argument("--bands", action="store_true", help="with --gpus N under torchrun: one lattice in N row bands (strong scaling) instead of N replicas")
    ap.add_argument("--bands-one-gpu", type=int, default=0, metavar="G", help="time the G-band algorithm band after band on one GPU next to sw_sweep")
    ap.add_argument("--ablation", action="store_true", help="time the paper's own labelling pipeline next to sw_label (SURVEY 8(f) row 4)")
    ap.add_argument("--no-per-config", action="store_true", help="skip the legs of the other BASELINE.json configs")
    ap.add_argument("--only-cubic", action="store_true", help="run the L=256 simple cubic leg alone (ncu captures of the k3_* kernels)")
    ap.add_argument("--no-cubic", action="store_true", help="skip the simple cubic lattice legs (SURVEY 8(f) row 2)")
    ap.add_argument("--no-other-betas", action="store_true", help="skip the beta = 0.40 / 0.50 legs of BASELINE.json configs[2]")
    ap.add_argument("--cpu-sweeps", type=int, default=3, help="oracle sweeps of the full lattice for cpu_baseline (0: L=4096 sample)")
    args = ap.parse_args(argv)
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        return run_reference(args)
    if args.ablation:
        return run_ablation(args)
    if args.only_cubic:
        return run_cubic_only(args)
    if args.bands:
        return run_bands(args)
    if args.bands_one_gpu > 1:
        return run_bands_one_gpu(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
