#!/usr/bin/env python
"""bench.py -- trial swaps/s of the SMC-X hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl reference]

A "step" is one Monte Carlo sweep of the whole hot path (LC origin, 8 colour
passes with tile staging / proposal / dE / accept / write-back, energy trace), plus a9 (pair-count
reduction -> energy + Warren-Cowley SRO) once every `sro_every` sweeps as the config prescribes and
at least once inside the timed region.  N = 1 times BASELINE.json configs[3] (BCC 800^3, 1.024e9
sites, the configuration the metric is quoted on).  N > 1 cuts that one lattice into N slabs along z, one per GPU,
with ghost layers exchanged after every colour pass (lattice parallelism; strong scaling); `--multi
replicas` runs N independent lattices instead (weak scaling, no data-path collective).

`--impl reference` times the CPU oracle (oracle/, test infrastructure) on the host cores for the
same metric; under torchrun only rank 0 works.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from dataclasses import replace  # noqa: E402

from smcx_inputs import get_config  # noqa: E402

ALGO_BYTES_PER_TRIAL = (686 + 250) / 128.0   # LIZ+ box read + modified box written per 128 trials
FALLBACK_HBM_GBS = 6650.0                    # B200_PROFILING.md fallback


def metric_name() -> str:
    try:
        return json.load(open(os.path.join(ROOT, "BASELINE.json")))["metric"]
    except Exception:
        return "trial swaps/sec on 1 B200 (1e9-site BCC, 4 species) and % of HBM roofline"


def measured_peak():
    try:
        return float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]), "measured"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback"


KERNEL_NAMES = {1: "sweep_warp_per_cell", 2: "sweep_thread_per_cell", 3: "sweep_thread_persistent", 4: "sweep_group_per_cell",
                5: "sweep_fcc_thread", 6: "sweep_local_warp", 7: "sweep_bcc4_thread"}
STORAGE_NAMES = {2: "2bit", 4: "4bit", 8: "u8"}
# Sources a kernel is compiled from: a number taken from an ncu capture (DRAM traffic, instruction counts per trial)
# is only reported next to live timings while these files are what they were at the capture.
KERNEL_SOURCES = {
    1: ["sweep_warp.cuh", "smcx_common.cuh"],
    2: ["sweep_thread.cuh", "sweep_warp.cuh", "smcx_common.cuh"],
    3: ["sweep_thread_sweep.cuh", "sweep_thread.cuh", "sweep_warp.cuh", "smcx_common.cuh"],
    4: ["sweep_group.cuh", "sweep_thread.cuh", "sweep_warp.cuh", "smcx_common.cuh"],
    5: ["sweep_fcc.cuh", "sweep_thread.cuh", "sweep_warp.cuh", "smcx_common.cuh"],
    6: ["sweep_local.cuh", "sweep_warp.cuh", "smcx_common.cuh"],
    7: ["sweep_bcc4.cuh", "sweep_fcc.cuh", "sweep_thread.cuh", "sweep_warp.cuh", "smcx_common.cuh"],
}
CAPTURES = os.path.join(ROOT, "profiles", "dram_traffic.csv")


def kernel_source_hash(kernel: int) -> str:
    import hashlib
    h = hashlib.sha256()
    for name in KERNEL_SOURCES[kernel]:
        with open(os.path.join(ROOT, "paper_2509_20949_b200", "csrc", name), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:12]


def load_capture(kernel: int, n_sites: int):
    """The committed ncu capture of this kernel on this workload (profiles/dram_traffic.csv), or (None, why)."""
    if not os.path.exists(CAPTURES):
        return None, "no capture file"
    want = kernel_source_hash(kernel)
    stale = None
    for line in open(CAPTURES):
        f = [x.strip() for x in line.split(",")]
        if len(f) < 8 or not f[0].isdigit() or int(f[0]) != kernel or int(f[1]) != n_sites:
            continue
        row = {"dram_bytes": float(f[2]), "source_hash": f[3], "alu_inst": float(f[4]), "wide": float(f[5]), "popc": float(f[6]),
               "capture": f[7]}
        if row["source_hash"] == want:
            return row, None
        stale = f"kernel sources changed since the capture {row['capture']} (hash {row['source_hash']} -> {want}): take a new one"
    return None, stale or "no capture of this kernel on this workload"


def alu_view(capture, trials_per_s: float, clocks: dict):
    """The integer ALU pipe is what binds the thread-per-cell kernels: instructions per trial on that pipe
    and the cycles an IMAD.WIDE / POPC holds it (profiles/r1_pipe_microbench.md), from the capture the sources match."""
    if capture is None:
        return None
    mhz = (clocks or {}).get("sm_max_mhz") or 1965.0
    peak = 148 * 4 * mhz * 1e6 / 2.0                      # ALU-pipe warp-instructions/s: 1 per 2 cycles per sub-partition
    inst = trials_per_s / 32.0 * capture["alu_inst"]
    busy = trials_per_s / 32.0 * (2.0 * capture["alu_inst"] + 2.6 * capture["wide"] + 1.0 * capture["popc"]) / (148 * 4 * mhz * 1e6)
    return {"bound": "alu", "achieved": inst, "peak": peak, "unit": "warp-inst/s", "frac": inst / peak,
            "alu_inst_per_trial": capture["alu_inst"], "pipe_busy_frac_with_wide_and_popc": busy,
            "note": f"whole-step trials/s; instruction counts from {capture['capture']}"}


def workload_string(cfg) -> str:
    lat = "BCC" if cfg.lattice == 0 else "FCC"
    return (f"{lat} {cfg.dims[0]}x{cfg.dims[1]}x{cfg.dims[2]} conventional cells ({cfg.n_sites} sites), "
            f"{cfg.n_species} species equiatomic, {cfg.n_shells}-shell int32 EPI in [-{cfg.amplitude},{cfg.amplitude}], "
            f"kT={cfg.kT_units / 10:g} meV, link cell {cfg.link_cell}, seed {cfg.seed}")


# --------------------------------------------------------------------------------------------
# clocks during the timed region (B200_PROFILING.md recipe)
# --------------------------------------------------------------------------------------------
class ClockSampler:
    QUERY = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
             "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.gpu}", f"--query-gpu={self.QUERY}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.lines:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); smax.append(float(f[2])); power.append(float(f[3]))
            except ValueError:
                continue
            for name, val in zip(names, f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


# --------------------------------------------------------------------------------------------
# CPU oracle timing (cpu_baseline and --impl reference)
# --------------------------------------------------------------------------------------------
def oracle_sample_config(cfg, max_sites: float = 8.3e6):
    """A bounded sample of the workload: same lattice type, species, EPI, kT, link cell, smaller box."""
    per_cell = 2 if cfg.lattice == 0 else 4
    edge = 16
    for e in (32, 48, 64, 96, 128, 160):
        if e ** 3 * per_cell <= max_sites:
            edge = e
    dims = tuple(min(d, edge) for d in cfg.dims)
    return replace(cfg, name=f"{cfg.name}@sample{edge}", dims=dims)


class OracleTimer:
    """The oracle as it stands (never tuned), one thread, on a bounded sample of the workload."""

    def __init__(self, cfg, max_sites: float = 8.3e6):
        import oracle
        self.sample = oracle_sample_config(cfg, max_sites)
        self.o = oracle.Oracle.from_config(self.sample)
        self.o.running_energy()
        self.t = 0

    def sweeps(self, n: int):
        t0 = time.perf_counter()
        for _ in range(n):
            if self.sample.anneal:
                self.o.set_temperature(self.sample.accept_table(self.t % self.sample.n_sweeps))
            self.o.sweep(1)
            self.t += 1
        return time.perf_counter() - t0

    def describe(self, n: int) -> str:
        d = self.sample.dims
        return (f"oracle (single thread, g++ -O2) on {d[0]}x{d[1]}x{d[2]} cells ({self.sample.n_sites} sites) "
                f"x {n} sweeps of the same workload (species, EPI, kT, link cell)")


def run_reference(args, cfg, rank):
    if rank != 0:
        return
    # size the per-step sample so that steps + warmup sweeps take about two minutes at ~2.5e6 trials/s
    budget_sites = 2.5e6 * 120.0 / max(1, args.steps + args.warmup)
    timer = OracleTimer(cfg, max_sites=min(8.3e6, max(7e4, budget_sites)))
    timer.sweeps(args.warmup)
    dt = timer.sweeps(args.steps)
    value = timer.sample.n_sites * args.steps / dt
    desc = timer.describe(args.steps)
    out = {
        "impl": "reference", "metric": metric_name(), "value": value, "unit": "trial swaps/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(1, args.steps),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
        "config": {"workload": workload_string(cfg), "note": "each step = 1 oracle sweep on the bounded sample"},
        "cpu_baseline": {"value": value, "unit": "trial swaps/s", "cores": 1, "kind": "oracle", "sample": desc,
                         "host_cores_available": os.cpu_count()},
        "e2e": {"value": value, "unit": "trial swaps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out))


# --------------------------------------------------------------------------------------------
# aggregation across ranks (testable with gloo on CPU)
# --------------------------------------------------------------------------------------------
def aggregate_over_ranks(local_ms: float, local_units: float, dist=None, device=None):
    """Whole-job throughput: units summed over ranks / max time over ranks.  Returns (value, max_ms)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return local_units / (local_ms * 1e-3), local_ms
    import torch
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    u = torch.tensor([local_units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(u.item()) / (float(t.item()) * 1e-3), float(t.item())


def replica_seed(base_seed: int, rank: int) -> int:
    """Independent replicas: rank r simulates the same workload with seed base + 7919 r."""
    return base_seed + 7919 * rank


# --------------------------------------------------------------------------------------------
# the CUDA arm
# --------------------------------------------------------------------------------------------
def run_ensemble(n_replicas: int, rounds: int = 20, sweeps_per_round: int = 10):
    """Temperature parallelism on one GPU: n_replicas of BASELINE.json config 2's lattice
    (BCC 64^3) on a ladder spaced as Eq. 7, rounds x (sweeps, replica-exchange round), device-timed."""
    import numpy as np
    import torch
    import paper_2509_20949_b200 as smcx
    from smcx_inputs import get_config, make_accept_table, replica_ladder

    cfg = get_config(2)
    kTs = replica_ladder(600, n_replicas, cfg.n_sites, 2.0 * float(np.sqrt(cfg.n_sites)))
    tabs = [make_accept_table(k) for k in kTs]
    ens = smcx.Ensemble(cfg.lattice, cfg.dims, cfg.n_species, cfg.n_shells, cfg.epi(), kTs, tabs,
                        [cfg.seed + 7919 * r for r in range(n_replicas)], cfg.seed)
    ens.run(rounds, sweeps_per_round)          # warm-up: captures the round graph
    ens.synchronize()
    l0 = ens.kernel_launches
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    ens.run(rounds, sweeps_per_round)
    b.record()
    ens.synchronize()
    torch.cuda.synchronize()
    ms = a.elapsed_time(b)
    st = ens.state()
    single = smcx.Lattice.from_config(cfg)
    single.sweep(rounds * sweeps_per_round)
    single.synchronize()
    a.record()
    single.sweep(rounds * sweeps_per_round)
    b.record()
    single.synchronize()
    torch.cuda.synchronize()
    ms1 = a.elapsed_time(b)
    n_sw = rounds * sweeps_per_round
    out = {"workload": f"{n_replicas} replicas of BCC 64^3 (524288 sites each), kT ladder {kTs[0]}..{kTs[-1]} (0.1 meV), "
                       f"{rounds} rounds x ({sweeps_per_round} sweeps + 1 exchange round)",
           "value": cfg.n_sites * n_replicas * n_sw / (ms * 1e-3), "unit": "trial swaps/s (all replicas)",
           "one_lattice_alone": cfg.n_sites * n_sw / (ms1 * 1e-3), "ms_per_round": ms / rounds,
           "exchange_accept_rate": float(st["accepted"].sum()) / max(1, int(st["attempted"].sum())),
           "gpu_launches": int(ens.kernel_launches - l0)}
    single.close()
    ens.close()
    return out


def _time_sweeps(lat, warm: int, sweeps: int) -> float:
    import torch
    lat.sweep(warm)
    lat.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    lat.sweep(sweeps)
    b.record()
    lat.synchronize()
    torch.cuda.synchronize()
    return a.elapsed_time(b) / sweeps


# Edge of the `paper_shaped_fcc` leg: FCC 640^3 = 1.05e9 sites, the size of the paper's per-GPU lattices (PAPER.md:141
# "1e9 sites per GPU", PAPER.md:165 1.07e9 sites).  tests/test_gpu_parity.py checks the same lattice.
PAPER_FCC_EDGE = 640


def run_paper_shaped_fcc(edge: int = PAPER_FCC_EDGE, sweeps: int = 10):
    """A lattice of the paper's own shape: FCC, five species in the proportions
    29/29/28/7/7 (reading S10), three shells, kT = 86 meV, synthetic EPI; the kernel AUTO picks (packed FCC kernel on
    4-bit storage) and, beside it, the sub-warp kernel on uint8 storage; device-timed."""
    import paper_2509_20949_b200 as smcx
    from smcx_inputs import composition_counts, make_accept_table, make_epi

    dims = (edge, edge, edge)
    peak, _ = measured_peak()
    out = {}
    for key, kernel in (("auto", smcx.KERNEL_AUTO), ("sub_warp", smcx.KERNEL_GROUP_PER_CELL)):
        lat = smcx.Lattice(smcx.FCC, dims, 5, 3, make_epi(3, 5, 400, 1006), make_accept_table(860), 1006, link_cell=4,
                           kT_units=860, kernel=kernel)
        lat.init_composition(composition_counts(lat.n_sites, (29, 29, 28, 7, 7)))
        ms = _time_sweeps(lat, 3, sweeps)
        out[key] = {"kernel": f"{KERNEL_NAMES[lat.kernel]}/{STORAGE_NAMES[lat.storage]}", "value": lat.n_sites / (ms * 1e-3),
                    "sweep_ms": ms}
        n_sites = lat.n_sites
        lat.close()
    v = out["auto"]["value"]
    return {"workload": f"FCC {edge}^3 conventional cells ({n_sites} sites), 5 species 29/29/28/7/7, 3-shell int32 EPI in "
                        f"[-400,400], kT=86 meV, link cell 4, seed 1006", "kernel": out["auto"]["kernel"],
            "value": v, "unit": "trial swaps/s", "sweep_ms": out["auto"]["sweep_ms"],
            "frac_of_hbm_roofline": v * ALGO_BYTES_PER_TRIAL / (peak * 1e9),
            "algorithmic_bytes_per_trial": ALGO_BYTES_PER_TRIAL,
            "device_bytes_per_trial_4bit": 8 * (0.5 + 0.5 * 36 / 64.0),
            "sub_warp_kernel": out["sub_warp"],
            "paper_h800_per_gpu": 3.5e9, "paper_note": "PAPER.md:130, EPI model on H800; other hardware and interactions: context"}


# Edge of the `local_energy_model` leg: FCC 256^3 = 6.7e7 sites, 32,768 link cells (warps) per colour pass, i.e. many waves
# of the 24 warps an SM holds; at 128^3 a pass is 1.15 waves (5.8-7.2e8 trials/s against 9.9e8).
LOCAL_EDGE = 256


def run_local_model(edge: int = LOCAL_EDGE, sweeps: int = 10):
    """The nonlinear local-energy model (reading S12; the role of the paper's qSRO model):
    FCC, five species 29/29/28/7/7, three shells, synthetic integer weights; every trial recomputes the local energies of
    the 86 sites its swap affects.  Device-timed."""
    import paper_2509_20949_b200 as smcx
    from smcx_inputs import composition_counts, make_accept_table, make_local_weights

    dims = (edge, edge, edge)
    w1, w2 = make_local_weights(3, 5, 200, 25, 1007)
    lat = smcx.Lattice(smcx.FCC, dims, 5, 3, w1, make_accept_table(2500), 1007, link_cell=4, kT_units=2500, local_quad=w2)
    lat.init_composition(composition_counts(lat.n_sites, (29, 29, 28, 7, 7)))
    ms = _time_sweeps(lat, 3, sweeps)
    acc = lat.stats()
    out = {"workload": f"FCC {edge}^3 conventional cells ({lat.n_sites} sites), 5 species 29/29/28/7/7, 3 shells, local-energy model "
                       f"eps = W1.n + n.W2.n with synthetic int32 weights, kT=250 meV, link cell 4, seed 1007",
           "kernel": "sweep_local_warp/u8", "value": lat.n_sites / (ms * 1e-3), "unit": "trial swaps/s", "sweep_ms": ms,
           "accept_rate": acc[2] / max(1, acc[1]),
           "paper_qsro_h800_per_gpu": 3.7e7, "paper_note": "PAPER.md:130, qSRO model on H800: another model and GPU, context only"}
    lat.close()
    return out


def run_bcc_five_species(edge: int = 800, sweeps: int = 10):
    """The graded lattice shape with FIVE species (more than the 2-bit kernels take): BCC edge^3, two shells, kT = 60 meV;
    the kernel AUTO picks (packed 4-bit BCC kernel, sweep_bcc4.cuh) and, beside it, the sub-warp kernel on uint8."""
    import paper_2509_20949_b200 as smcx
    from smcx_inputs import make_accept_table, make_epi

    peak, _ = measured_peak()
    out = {}
    for key, kernel in (("auto", smcx.KERNEL_AUTO), ("sub_warp", smcx.KERNEL_GROUP_PER_CELL)):
        lat = smcx.Lattice(smcx.BCC, (edge, edge, edge), 5, 2, make_epi(2, 5, 300, 1008), make_accept_table(600), 1008,
                           link_cell=4, kT_units=600, kernel=kernel)
        ms = _time_sweeps(lat, 3, sweeps)
        out[key] = {"kernel": f"{KERNEL_NAMES[lat.kernel]}/{STORAGE_NAMES[lat.storage]}", "value": lat.n_sites / (ms * 1e-3), "sweep_ms": ms}
        n_sites = lat.n_sites
        lat.close()
    v = out["auto"]["value"]
    return {"workload": f"BCC {edge}^3 conventional cells ({n_sites} sites), 5 species equiatomic, 2-shell int32 EPI in [-300,300], "
                        f"kT=60 meV, link cell 4, seed 1008", "kernel": out["auto"]["kernel"], "value": v, "unit": "trial swaps/s",
            "sweep_ms": out["auto"]["sweep_ms"], "frac_of_hbm_roofline": v * ALGO_BYTES_PER_TRIAL / (peak * 1e9),
            "sub_warp_kernel": out["sub_warp"]}


def run_largest_single_gpu(sweeps: int = 20):
    """BASELINE.json configs[4]: BCC 2000^3, 1.6e10 sites (4 GB in 2-bit storage), device-timed."""
    import paper_2509_20949_b200 as smcx

    cfg = get_config(5)
    peak, _ = measured_peak()
    lat = smcx.Lattice.from_config(cfg)
    ms = _time_sweeps(lat, 3, sweeps)
    v = cfg.n_sites / (ms * 1e-3)
    out = {"workload": workload_string(cfg), "config_id": 5, "kernel": f"{KERNEL_NAMES[lat.kernel]}/{STORAGE_NAMES[lat.storage]}",
           "sweeps": sweeps, "value": v, "unit": "trial swaps/s", "sweep_ms": ms,
           "frac_of_hbm_roofline": v * ALGO_BYTES_PER_TRIAL / (peak * 1e9)}
    lat.close()
    return out


def run_lattice_parallel_one_gpu(cfg, sweeps: int = 10, whole_sweep_ms=None):
    """Lattice parallelism with every slab on this one GPU: the workload cut into
    2 and 4 slabs with ghost layers, messages as device-to-device copies, with and without computation-communication
    overlap.  Measures what the decomposition itself costs (split launches, messages, event ordering); the slabs
    share one GPU, so this is not a scaling number."""
    import paper_2509_20949_b200 as smcx

    out = {"workload": workload_string(cfg), "note": "all slabs on one GPU: cost of the decomposition, not scaling",
           "undivided_sweep_ms": whole_sweep_ms, "runs": []}
    for n_slabs, overlap in ((2, 1), (4, 1), (4, 2), (4, 0)):
        g = smcx.DomainGroup.from_config(cfg, n_slabs, overlap=overlap)
        ms = _time_sweeps(g, 3, sweeps)
        b0 = g.message_bytes
        g.sweep(1)
        g.synchronize()
        out["runs"].append({"slabs": n_slabs, "mode": {0: "pass, then copy", 1: "boundary row (side stream, message fused into its kernel) and the other rows concurrently on disjoint SMs",
                                                        2: "boundary row first, message copied on a second stream"}[overlap],
                            "fused_messages_per_sweep": int(g.fused_messages // max(1, g.stats()[0])), "sweep_ms": ms, "value": cfg.n_sites / (ms * 1e-3),
                            "unit": "trial swaps/s", "message_bytes_per_sweep": int(g.message_bytes - b0),
                            "vs_undivided": (whole_sweep_ms / ms) if whole_sweep_ms else None})
        g.close()
    # connected slabs (the one-slab-per-process path of `--gpus N`) with both slabs in this process: messages written by
    # the sweep kernels into the neighbour's storage, ordering by flags and stream memory waits, no events, no copies
    import torch
    kw = dict(lattice=cfg.lattice, dims=cfg.dims, n_species=cfg.n_species, n_shells=cfg.n_shells, epi=cfg.epi(),
              accept=cfg.accept_table(0), seed=cfg.seed, link_cell=cfg.link_cell, kT_units=cfg.kT_at(0))
    streams = [torch.cuda.Stream() for _ in range(2)]
    slabs = [smcx.Domain(2, r, stream=streams[r], **kw) for r in range(2)]
    for r in range(2):
        slabs[r].connect(slabs[1 - r], slabs[1 - r])

    def step(n):
        for _ in range(n):
            for sl in slabs:
                sl.sweep_connected(1)
    step(3)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for st in streams:
        st.wait_event(a)
    step(sweeps)
    for st in streams:
        torch.cuda.current_stream().wait_stream(st)
    b.record()
    torch.cuda.synchronize()
    ms = a.elapsed_time(b) / sweeps
    out["runs"].append({"slabs": 2, "mode": "connected slabs (flags + stream memory waits, messages fused), both in this process",
                        "fused_messages_per_sweep": 16, "sweep_ms": ms, "value": cfg.n_sites / (ms * 1e-3), "unit": "trial swaps/s",
                        "message_bytes_per_sweep": None, "vs_undivided": (whole_sweep_ms / ms) if whole_sweep_ms else None})
    for sl in slabs:
        sl.close()
    return out


def run_slabs(args, cfg, rank, world, local_rank):
    """N > 1: the paper's lattice parallelism: the ONE lattice of the config cut into N slabs along z, one
    per GPU / rank, ghost layers exchanged after every colour pass with torch.distributed send/recv (NCCL), the
    boundary row of a pass first so that its message overlaps the other rows.  Strong scaling: the total
    work is fixed.  Results are those of the undivided lattice bit for bit (tests/test_gpu_domains.py)."""
    import torch
    import torch.distributed as dist
    from paper_2509_20949_b200 import distributed

    local_rank = local_rank % torch.cuda.device_count()      # several ranks may share a GPU (one-GPU test runs of this path)
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if not dist.is_initialized():
        if args.dist_backend == "nccl":
            dist.init_process_group("nccl", device_id=dev)
        else:
            dist.init_process_group(args.dist_backend)

    def barrier():
        dist.barrier()
        torch.cuda.synchronize()

    kw = dict(lattice=cfg.lattice, dims=cfg.dims, n_species=cfg.n_species, n_shells=cfg.n_shells, epi=cfg.epi(),
              accept=cfg.accept_table(0), seed=cfg.seed, link_cell=cfg.link_cell, kT_units=cfg.kT_at(0),
              kernel=args.kernel, storage=args.storage, device=local_rank)
    transport = args.transport
    slab = None
    if transport == "ipc":
        # ghost layers by peer stores from inside the sweep kernels, signalled through device flags (one node)
        try:
            slab = distributed.ConnectedSlabRank(rank, world, dist=dist, **kw)
        except Exception as exc:                     # e.g. no peer access between two GPUs: every rank fails alike at connect
            if rank == 0:
                print(f"bench.py: connected slabs unavailable ({exc}); using NCCL messages", file=sys.stderr)
            transport = "nccl"
    if slab is None:
        slab = distributed.SlabRank(rank, world, dist=dist, overlap=not args.no_overlap, **kw)
    slab.sweep(args.warmup)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.25)
    launches0 = slab.domain.kernel_launches
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    a.record()
    slab.sweep(args.steps)
    b.record()
    barrier()
    total_ms = a.elapsed_time(b)
    clocks = sampler.stop()
    launches = slab.domain.kernel_launches - launches0
    owned = float(slab.domain.info["owned_sites"])
    value, max_ms = aggregate_over_ranks(total_ms, owned * args.steps, dist, dev)
    # end to end: every rank uploads its window of the host array, K x (table up, sweep, energy back), owned layers down
    host = torch.empty(cfg.n_sites, dtype=torch.uint8).pin_memory().numpy()
    host[:] = 0
    slab.domain.species_into(host)
    whole = torch.from_numpy(host).to(dev)
    dist.all_reduce(whole)                       # owned layers are disjoint: the sum is the whole lattice
    host[:] = whole.cpu().numpy()
    del whole
    e2e_steps = min(args.steps, 200)
    table = cfg.accept_table(0)
    barrier()
    t0 = time.perf_counter()
    slab.domain.set_species(host)
    first = slab.domain.stats()[0]
    for t in range(e2e_steps):
        slab.domain.set_temperature(cfg.kT_at(0), table)
        slab.sweep(1)
        slab.domain.energy_trace(first + t, 1)
    slab.domain.species_into(host)
    counts = slab.pair_counts()
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_value, _ = aggregate_over_ranks(e2e_s * 1e3, owned * e2e_steps, dist, dev)
    window = slab.domain.info["z_layers"] * cfg.n_sites // cfg.dims[2]
    if rank == 0:
        peak, peak_kind = measured_peak()
        launch_ms = max_ms / args.steps / 8.0
        achieved = ALGO_BYTES_PER_TRIAL * (cfg.n_sites / 8.0 / world) / (launch_ms * 1e-3) / 1e9
        out = {
            "metric": metric_name(), "value": value, "unit": "trial swaps/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": max_ms / args.steps, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "int32", "data": "synthetic",
            "config": {"workload": workload_string(cfg), "config_id": args.config,
                       "step": "1 sweep of the one lattice = per GPU a window shift + 8 x (colour pass of its slab, ghost-layer message)",
                       "parallelism": (f"lattice parallelism: {world} slabs along z, one per GPU, ghost layers written by the sweep "
                                       "kernels into the neighbour GPU's memory (CUDA IPC peer stores), signalled by device flags"
                                       if transport == "ipc" else
                                       f"lattice parallelism: {world} slabs along z, one per GPU, ghost layers over NCCL send/recv, "
                                       f"overlap {'on' if not args.no_overlap else 'off'}"),
                       "l2": "slab windows larger than the 126 MB L2 at the graded size; no flush"},
            "pct_of_hbm_roofline": 100.0 * (value / world) * ALGO_BYTES_PER_TRIAL / (peak * 1e9),
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": None, "traffic_note": "multi-GPU run: no ncu capture (profiles/ hold the single-GPU ones)",
                         "peak_kind": peak_kind, "kernel": KERNEL_NAMES.get(args.kernel, "auto"),
                         "what": "per GPU: algorithmic bytes of one colour pass of a slab / (step time / 8), message wait included",
                         "algorithmic_bytes_per_trial": ALGO_BYTES_PER_TRIAL, "launch_ms": launch_ms},
            "e2e": {"value": e2e_value, "unit": "trial swaps/s", "h2d_bytes_per_step": (window + e2e_steps * table.nbytes) / e2e_steps,
                    "d2h_bytes_per_step": (owned + e2e_steps * 8 + counts.nbytes) / e2e_steps, "steps": e2e_steps,
                    "what": "per rank: smcx_domain_set_species(host) + steps x (table up, sweep with messages, energy back) + "
                            "smcx_domain_species(host) + pair counts, wall clock, max over ranks"},
            "message_bytes_per_step_per_gpu": slab.message_bytes / max(1, args.warmup + args.steps + e2e_steps),
            "gpu_launches": int(launches), "clocks": clocks,
        }
        print(json.dumps(out))
    slab.close()
    dist.barrier()
    dist.destroy_process_group()


def run_cuda(args, cfg, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    import paper_2509_20949_b200 as smcx

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1 and not dist.is_initialized():
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sro_every = cfg.sro_every if cfg.sro_every > 0 else 1000
    lat = smcx.Lattice.from_config(cfg, seed=replica_seed(cfg.seed, rank), device=local_rank,
                                   kernel=args.kernel, storage=args.storage)
    tables = None
    if cfg.anneal:
        tables = [(cfg.kT_at(t), cfg.accept_table(t)) for t in range(min(cfg.n_sweeps, args.steps + args.warmup))]

    def one_step(t):
        if tables is not None:
            kT, tab = tables[t % len(tables)]
            lat.set_temperature(kT, tab)
        lat.sweep(1)

    if tables is None:
        lat.sweep(args.warmup)        # same call as the timed region: the sweep graph is captured here, not there
    else:
        for t in range(args.warmup):
            one_step(t)
    lat.sro()
    barrier()

    # ---- device-resident timing -----------------------------------------------------------
    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.25)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    launches0 = lat.kernel_launches
    barrier()
    ev[0].record()
    sweep_ms = 0.0
    sro_ms = 0.0
    done = 0
    n_sro = 0
    while done < args.steps:
        chunk = min(sro_every - (done % sro_every), args.steps - done)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        if tables is None:
            lat.sweep(chunk)          # fixed temperature: one call, replayed from the captured sweep graph
        else:
            for t in range(chunk):
                one_step(args.warmup + done + t)
        b.record()
        done += chunk
        c0 = torch.cuda.Event(enable_timing=True); c1 = torch.cuda.Event(enable_timing=True)
        c0.record()
        if done % sro_every == 0 or done == args.steps:
            alpha, counts = lat.sro()      # a9: synchronises
            n_sro += 1
        c1.record()
        torch.cuda.synchronize()
        sweep_ms += a.elapsed_time(b)
        sro_ms += c0.elapsed_time(c1)
    ev[1].record()
    barrier()
    total_ms = ev[0].elapsed_time(ev[1])
    launches = lat.kernel_launches - launches0
    clocks = sampler.stop()

    trials = float(cfg.n_sites) * args.steps
    value, max_ms = aggregate_over_ranks(total_ms, trials, dist if world > 1 else None, dev)

    # ---- end to end through the C ABI with host buffers -------------------------------------
    # one job = upload the lattice from pinned host memory, K x (upload that sweep's threshold
    # table, sweep, read the sweep's energy back), download the lattice, SRO.
    host_species = torch.empty(cfg.n_sites, dtype=torch.uint8).pin_memory().numpy()
    lat.species(out=host_species)
    e2e_steps = min(args.steps, 200)   # one job: the lattice goes up and comes back once, the steps in between
    table = cfg.accept_table(0)
    barrier()
    t0 = time.perf_counter()
    lat.set_species(host_species)
    first = lat.stats()[0]
    for t in range(e2e_steps):
        if tables is not None:
            kT, table = tables[t % len(tables)]
        lat.set_temperature(cfg.kT_at(0) if tables is None else kT, table)
        lat.sweep(1)
        lat.energy_trace(first + t, 1)
    lat.species(out=host_species)
    lat.sro()
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_value, _ = aggregate_over_ranks(e2e_s * 1e3, float(cfg.n_sites) * e2e_steps, dist if world > 1 else None, dev)
    h2d = (cfg.n_sites + e2e_steps * table.nbytes) / e2e_steps
    d2h = (cfg.n_sites + e2e_steps * 8 + 2 * counts.nbytes) / e2e_steps

    if rank == 0:
        peak, peak_kind = measured_peak()
        # dominant kernel: one colour pass = n_sites/8 trials per launch, 8 launches per sweep -- or, where the library
        # pipelines the eight passes in ONE launch (sweep_thread_whole_sweep: 3 launches per sweep instead of 9), the whole
        # sweep = n_sites trials per launch
        passes_per_launch = 8 if (lat.kernel == 3 and launches < 6 * args.steps) else 1
        launch_ms = sweep_ms / args.steps * passes_per_launch / 8.0
        achieved = ALGO_BYTES_PER_TRIAL * (cfg.n_sites * passes_per_launch / 8.0) / (launch_ms * 1e-3) / 1e9
        # DRAM bytes per launch and instruction counts come from an ncu capture: reported only while the kernel's
        # sources are what they were when it was taken, null (with the reason) otherwise
        capture, capture_note = load_capture(lat.kernel, cfg.n_sites)
        traffic = capture["dram_bytes"] if capture else None
        dev_bytes = cfg.n_sites * {2: 0.25, 4: 0.5, 8: 1.0}[lat.storage]
        frac = achieved / peak
        out = {
            "metric": metric_name(), "value": value, "unit": "trial swaps/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": max_ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int32", "data": "synthetic",
            "config": {
                "workload": workload_string(cfg), "config_id": args.config,
                "step": f"1 sweep = {'1 launch of all 8 colour passes' if passes_per_launch == 8 else '8 colour-pass launches'} + trace; pair-count/SRO reduction every {sro_every} sweeps "
                        f"and once at the end ({n_sro} inside the timed region)",
                "kernel": f"{KERNEL_NAMES[lat.kernel]}/{STORAGE_NAMES[lat.storage]}",
                "l2": ("lattice (%.0f MB in device storage) larger than the 126 MB L2; no flush" % (dev_bytes / 1e6))
                      if dev_bytes > 126e6 else
                      ("lattice (%.1f MB in device storage) fits the 126 MB L2 and stays resident between sweeps; no flush: "
                       "this configuration is latency-bound, not a bandwidth measurement" % (dev_bytes / 1e6)),
                "parallelism": "replicas only" if world > 1 else "single GPU",
            },
            "pct_of_hbm_roofline": 100.0 * (value / world) * ALGO_BYTES_PER_TRIAL / (peak * 1e9),
            "sweep_ms": sweep_ms / args.steps, "sro_ms_each": sro_ms / max(1, n_sro),
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": frac,
                         "traffic": traffic, "traffic_note": capture_note, "peak_kind": peak_kind,
                         "kernel": "sweep_thread_whole_sweep" if passes_per_launch == 8 else KERNEL_NAMES[lat.kernel],
                         "colour_passes_per_launch": passes_per_launch,
                         "what": "achieved = ALGORITHMIC bytes (uint8, SURVEY.md 8(d)) per launch / measured launch time, as "
                                 "north_star declares the roofline; the bytes the kernel really moves are in `dram`",
                         "algorithmic_bytes_per_trial": ALGO_BYTES_PER_TRIAL, "launch_ms": launch_ms,
                         "north_star_target_frac": 0.5, "target_met": bool(frac >= 0.5),
                         "schedule_ceiling_frac": (0.346 if lat.kernel == 3 else None),
                         "schedule_ceiling_note": "DESIGN.md 7: the trial S3/S4 prescribe costs >= 120 ALU-pipe cycles per warp-trial "
                                                  "(Philox4x32-10 alone is 20 % of a pass, measured by ablation), i.e. 0.413 ms per colour "
                                                  "pass = 34.6 % of this roofline with that pipe 100 % busy; the kernel is ALU-bound "
                                                  "(see alu_view), HBM runs at 10 % of peak (see dram)"},
            # what the kernel moves (packed storage): measured DRAM bytes per launch / live launch time
            "dram": ({"bytes_per_launch": traffic, "achieved_gbs": traffic / (launch_ms * 1e-3) / 1e9,
                      "frac_of_peak": traffic / (launch_ms * 1e-3) / 1e9 / peak, "source": capture["capture"]}
                     if capture else None),
            "alu_view": alu_view(capture, value / world, clocks),
            "e2e": {"value": e2e_value, "unit": "trial swaps/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": e2e_steps,
                    "what": "smcx_set_species(host) + steps x (smcx_set_temperature(host table) + smcx_sweep(1) + "
                            "smcx_energy_trace read) + smcx_species(host) + smcx_sro, wall clock"},
            "gpu_launches": int(launches), "clocks": clocks,
        }
        if not args.no_cpu_baseline and world == 1:
            timer = OracleTimer(cfg)
            n_or = 3
            dt = timer.sweeps(n_or)
            v, desc = timer.sample.n_sites * n_or / dt, timer.describe(n_or)
            out["cpu_baseline"] = {"value": v, "unit": "trial swaps/s", "cores": 1, "kind": "oracle", "sample": desc,
                                   "host_cores_available": os.cpu_count()}
        if args.ensemble > 1 and world == 1:
            lat.close()
            out["temperature_parallel"] = run_ensemble(args.ensemble)
            if args.fcc_edge > 0:
                out["paper_shaped_fcc"] = run_paper_shaped_fcc(args.fcc_edge)
            if args.largest and args.config != 5:
                out["largest_single_gpu"] = run_largest_single_gpu()
            if args.local_edge > 0:
                out["local_energy_model"] = run_local_model(args.local_edge)
            if args.fcc_edge > 0:
                out["bcc_five_species"] = run_bcc_five_species()
            if args.slabs_leg and cfg.dims[2] // cfg.link_cell >= 16:
                out["lattice_parallel_one_gpu"] = run_lattice_parallel_one_gpu(cfg, whole_sweep_ms=sweep_ms / args.steps)
        print(json.dumps(out))
    lat.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config 1..5 (default: 4, the graded one)")
    ap.add_argument("--kernel", type=int, default=0, help="0 auto, 1 warp-per-cell, 2 thread-per-cell, 3 thread-per-cell persistent, 4 sub-warp group per cell, 5 packed FCC thread-per-cell")
    ap.add_argument("--storage", type=int, default=0, help="0 auto, 2 packed 2-bit, 4 packed 4-bit, 8 uint8")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--fcc-edge", type=int, default=PAPER_FCC_EDGE,
                    help="with --ensemble: also time the sub-warp kernel on an FCC lattice of the paper's shape, this many "
                         "conventional cells per edge (0: skip)")
    ap.add_argument("--no-largest", dest="largest", action="store_false",
                    help="skip the BCC 2000^3 (1.6e10 sites) leg that the default run adds as `largest_single_gpu`")
    ap.add_argument("--local-edge", type=int, default=LOCAL_EDGE,
                    help="with --ensemble: also time the nonlinear local-energy model on an FCC lattice of this edge (0: skip)")
    ap.add_argument("--no-slabs-leg", dest="slabs_leg", action="store_false",
                    help="skip the `lattice_parallel_one_gpu` leg (the workload cut into 2 / 4 slabs on this one GPU)")
    ap.add_argument("--multi", default="slabs", choices=["slabs", "replicas"],
                    help="N > 1: `slabs` = the one lattice cut into N slabs, one per GPU (lattice parallelism, strong scaling); "
                         "`replicas` = N independent lattices (weak scaling)")
    ap.add_argument("--dist-backend", default="nccl", choices=["nccl", "gloo"],
                    help="--multi slabs: torch.distributed backend for handles, barriers and reductions (gloo: ranks that share a GPU)")
    ap.add_argument("--transport", default="ipc", choices=["ipc", "nccl"],
                    help="--multi slabs: how ghost layers travel: `ipc` = peer stores from the sweep kernels + device flags "
                         "(connected slabs, one node), `nccl` = torch.distributed send/recv")
    ap.add_argument("--no-overlap", action="store_true", help="--multi slabs: send the ghost layers after the whole pass")
    ap.add_argument("--source-hash", action="store_true", help="print the source hash of every kernel (for profiles/dram_traffic.csv) and exit")
    ap.add_argument("--ensemble", type=int, default=128,
                    help="also time a replica-exchange ensemble of this many BCC 64^3 replicas (0: skip)")
    args = ap.parse_args()
    if args.source_hash:
        for k in sorted(KERNEL_SOURCES):
            print(k, KERNEL_NAMES[k], kernel_source_hash(k))
        return
    args.warmup = max(args.warmup, 3) if args.impl == "cuda" else args.warmup
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    cfg = get_config(args.config)
    if args.impl == "reference":
        run_reference(args, cfg, rank)
        return
    if world > 1 and args.multi == "slabs":
        run_slabs(args, cfg, rank, world, local_rank)
        return
    run_cuda(args, cfg, rank, world, local_rank)


if __name__ == "__main__":
    main()
