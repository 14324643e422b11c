#!/usr/bin/env python
"""bench.py — spin flips per ns of the double-checkerboard Metropolis sweep (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--layout int8|bits] [--tile 32|64] [--k 1|4|16] [--L 16384] [--no-extras]

One "step" = one outer pass of the whole hot path (colour-0 launch + colour-1 launch, k inner
sweeps each) over the 2D L=16384 lattice of BASELINE.json config 3 (seed 3, beta = 0.4406868),
spins resident in HBM.  `value` = attempted flips per ns = K * k * L^2 / t (time per attempted
flip, measurement of E/M excluded).  Multi-GPU (`--gpus N` under torchrun): the path does not shard
by contract (north_star: one GPU), so N ranks run N independent replicas ("replicas only", DESIGN.md
§8) and `value` is the aggregate.  `--impl reference` times the CPU oracle (test infrastructure) on a
bounded sample of the same workload; it is the only place besides `cpu_baseline` that touches oracle/.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import ising_workloads as W  # noqa: E402

METRIC = "spin flips/ns (2D Ising L=16384, beta_c)"
UNIT = "flips/ns"


def algorithmic_bytes_per_flip(tile: int, k: int, layout: str, L: int = 0) -> float:
    """read s(1 + 2*dim/T) + write s per site per pass, / k; s = 1 B int8, 1/8 B bits.
    Plain checkerboard (tile == L, row a8): each half-sweep reads every site and writes the updated half: 3 s per flip."""
    s = 1.0 if layout == "int8" else 0.125
    if tile in (0, L):
        return 3.0 * s
    return s * (2.0 + 4.0 / tile) / k


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)", float(d.get("sm_max_mhz", 1965.0))
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)", 1965.0


FP_FILES = {   # the device sources a kernel family is built from
    "flow": ("philox.cuh", "planes_common.cuh", "tile_planes_device.cuh", "flow_planes_device.cuh"),
    "tile": ("philox.cuh", "planes_common.cuh", "tile_planes_device.cuh", "flow_planes_device.cuh"),
    "grid": ("philox.cuh", "planes_common.cuh", "tile_planes_device.cuh", "grid_planes_device.cuh"),
}


def kernel_fingerprint(family: str = "grid") -> str:
    """sha1 (12 hex digits) over the sources of a kernel family: an ncu figure quoted below is only printed while the
    kernel it was captured from is the kernel being timed."""
    import hashlib
    h = hashlib.sha1()
    for n in FP_FILES[family]:
        h.update(open(os.path.join(ROOT, "paper_1006_3865_b200", "csrc", n), "rb").read())
    return h.hexdigest()[:12]


# From the committed ncu captures, per PHASE (one coarse colour of one pass = one launch of k_tile_planes, or a sixth of
# the captured 3-pass launch of the persistent k_flow_planes): DRAM bytes read + written, and executed warp-instructions.
# The grid-resident kernel (lattice on chip for the whole call) touches DRAM once per CALL: its entries hold the bytes and
# the instructions of a call's load + store ("*_call") and the instructions of one pass, separated by two captures of 8 and
# 16 passes; a phase of a K-pass call is then (call + K * pass) / 2K.
# Keyed by (rng, layout, tile, k, kernel family); "fp" = kernel_fingerprint(family) of the sources they were captured from.
NCU = {
    ("planes", "int8", 64, 1, "flow"): {"traffic": (803.28e6 + 757.91e6) / 6, "warp_instr": 219.54e6 / 6, "fp": "7acfaaf12164", "source": "profiles/r02c_flow_planes_i8.md"},
    ("planes", "int8", 32, 1, "flow"): {"traffic": (803.52e6 + 798.38e6) / 6, "warp_instr": 246.42e6 / 6, "fp": "7acfaaf12164", "source": "profiles/r02c_flow_planes_i8.md"},
    ("planes", "int8", 64, 1, "tile"): {"traffic": 138.44e6 + 80.40e6, "warp_instr": 33.73e6, "fp": "7acfaaf12164", "source": "profiles/r02c_flow_planes_i8.md"},
    ("planes", "int8", 64, 1, "grid"): {"traffic_call": 277.03e6 + 222.71e6, "warp_instr_call": 480.83e6 - 8 * 58.560e6, "warp_instr_pass": 58.560e6,
                                        "pipes_16_passes": {"alu": 0.617, "fmaheavy": 0.598, "issue_active": 0.549},
                                        "fp": "c1c009a23ee4", "source": "profiles/r02e_grid_planes_L16384.md"},
    ("planes", "int8", 32, 1, "grid"): {"traffic_call": 321.08e6 + 255.54e6, "warp_instr_call": 581.98e6 - 8 * 70.146e6, "warp_instr_pass": 70.146e6,
                                        "pipes_16_passes": {"alu": 0.615, "fmaheavy": 0.610, "issue_active": 0.585},
                                        "fp": "c1c009a23ee4", "source": "profiles/r02e_grid_planes_L16384.md"},
}


def ncu_per_phase(entry, steps: int):
    """(DRAM bytes, warp-instructions) of one phase of a `steps`-pass call from an NCU entry, or (None, None)."""
    if entry is None:
        return None, None
    if "traffic_call" in entry:
        return entry["traffic_call"] / (2 * steps), (entry["warp_instr_call"] + steps * entry["warp_instr_pass"]) / (2 * steps)
    return entry["traffic"], entry["warp_instr"]


# Issue slots of the GPU: 148 SMs x 4 schedulers, one warp-instruction per cycle at sm_max_mhz.
def issue_peak_gips(sm_mhz: float) -> float:
    return 148 * 4 * sm_mhz * 1e6 / 1e9


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._pump, daemon=True).start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def wait_first_row(self, timeout: float) -> None:
        """nvidia-smi needs a few hundred ms before its first row: do not start the timed region without one."""
        t = time.time()
        while self.proc is not None and not self.rows and time.time() - t < timeout:
            time.sleep(0.02)

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for r in self.rows if t0 - 0.05 <= r[0] <= t1 + 0.15]
        if len(rows) < 2:            # a timed region shorter than the sampling period: the rows around it
            rows = [r for r in self.rows if t0 - 0.3 <= r[0] <= t1 + 0.3] or self.rows
        for _, line in rows:
            f = [x.strip() for x in line.split(",")]
            try:
                sm.append(float(f[0])); mx = float(f[1])
            except Exception:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


def oracle_flips_per_ns(L: int, tile: int, k: int, passes: int, rng: str = "planes"):
    """Time the CPU oracle as it stands: `passes` outer passes on an L x L lattice, 1 core."""
    from oracle import oracle as O
    O.build()
    o = O.Oracle(2, L, seed=3, rng=rng)
    t0 = time.perf_counter()
    o.sweep(W.BETA_C_2D, passes, tile, k)
    dt = time.perf_counter() - t0
    return passes * k * L * L / dt / 1e9, dt


def run_reference(a, rank: int, world: int) -> None:
    if rank != 0:
        return
    Ls = 4096                                   # bounded sample: 1/16 of the L=16384 sites per step
    per_step = []
    for i in range(a.warmup + a.steps):
        v, dt = oracle_flips_per_ns(Ls, a.tile, a.k, 1, a.rng)
        if i >= a.warmup:
            per_step.append(dt)
    tot = sum(per_step)
    val = a.steps * a.k * Ls * Ls / tot / 1e9
    sample = f"each step = one outer pass (tile {a.tile}, k {a.k}, beta_c) of a {Ls}x{Ls} hot-start lattice, seed 3"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": a.gpus, "steps": a.steps,
            "warmup": a.warmup, "ms_per_step": 1e3 * tot / a.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int8", "data": "synthetic",
            "config": {"workload": f"BASELINE config 3: 2D Ising L=16384 {a.layout} tile={a.tile} k={a.k} (oracle on a bounded sample)"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def aggregate_replicas(ms_local: float, world: int, steps: int, k: int, L: int, dist=None, device="cpu"):
    """'Replicas only': every rank ran the same independent workload; the job's time is the MAX
    over ranks and the job's work is the sum.  Returns (ms, flips_per_ns)."""
    ms = ms_local
    if dist is not None:
        import torch
        t = torch.tensor([ms_local], device=device, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    return ms, world * steps * k * L * L / (ms * 1e6)


def selftest_ranks(rank: int, world: int) -> None:
    """CPU check of the multi-rank plumbing (gloo, no GPU): rank r pretends to have taken (1 + r) ms."""
    import torch.distributed as dist
    dist.init_process_group("gloo")
    dist.barrier()
    ms, value = aggregate_replicas(1.0 + rank, world, steps=2, k=1, L=1000, dist=dist)
    assert ms == float(world), (ms, world)
    if rank == 0:
        print(json.dumps({"selftest": "ranks", "n_gpus": world, "ms": ms, "value": value, "scaling": "weak"}), flush=True)
    dist.destroy_process_group()


JIT = "auto"     # --jit: run-time specialisation of the planes kernel (ising_set_jit)
FORCE = 0        # --force-path: ising_force_path (0 automatic, 2 a launch per colour, 3 no data-flow kernel, 4 no on-chip kernels)


def time_variant(P, torch, L, layout, tile, k, steps, warmup, sampler=None, rng="planes", min_seconds=0.0, max_reps=1, force=None):
    """Device-timed throughput of one (rng, layout, tile, k) variant; returns dict.

    One repetition = one `ising_sweep(steps)` call = exactly `steps` outer passes (2 launches each, no host sync inside),
    bracketed by CUDA events on the library's stream.  The repetition is repeated back to back until `min_seconds` of GPU
    time have elapsed (at most `max_reps` times): `ms` is the MEDIAN repetition, `ms_min` / `ms_max` the spread.  The
    clock sampler (if any) runs from before the warm-up to after the last repetition, so that it has rows however short a
    repetition is (20 steps are 2.4 ms)."""
    g = P.Ising(2, L, seed=3, rng=rng)
    # the library's AUTO rule (specialise calls of >= 2^27 attempted flips), decided here for the timed call so that
    # the warm-up call, which is shorter, already compiles the kernel the timed call will use
    # (lattices small enough for the resident kernels stay on AUTO: they serve them)
    # Lattices that live on chip for a whole call (cluster / grid resident kernels: at most two jobs of a colour per warp of the
    # GPU) stay on the library's AUTO rule: it chooses between the producer / consumer form and the specialised kernel.
    onchip = tile in (32, 64) and (L // tile) ** 2 // 2 // (64 // tile) <= 148 * 20 * 2 and steps >= 2
    if not onchip:
        g.set_jit("on" if JIT == "on" or (JIT == "auto" and steps * k * L * L >= 2 ** 27) else "off")
    else:
        g.set_jit(JIT)
    if tile in (32, 64) and steps >= 2:
        # the same call once before: which kernel serves a call depends on its length (a lattice is put on chip only for a
        # call long enough to pay for it), so only the same call compiles, outside the timed region, what the timed call runs
        warmup = max(warmup, steps)
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    if force if force is not None else FORCE:
        g.force_path(force if force is not None else FORCE)
    if sampler:
        sampler.start()
    g.sweep(W.BETA_C_2D, warmup, tile, k)
    g.synchronize()
    torch.cuda.synchronize()
    if sampler:
        sampler.wait_first_row(3.0)
    n0 = P.ising_kernel_launches()
    t0 = time.time()
    events, total, reps = [], 0.0, 0
    while True:
        batch = []
        for _ in range(1 if reps == 0 else min(max_reps - reps, max(1, int(0.25 * reps / max(total, 1e-6))))):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            g.sweep(W.BETA_C_2D, steps, tile, k)        # K passes = 2K launches, no host sync in between
            e1.record()
            batch.append((e0, e1))
        torch.cuda.synchronize()
        ms_batch = [a.elapsed_time(b) for a, b in batch]
        events += ms_batch
        total += sum(ms_batch) / 1e3
        reps += len(batch)
        if total >= min_seconds or reps >= max_reps:
            break
    t1 = time.time()
    launches = (P.ising_kernel_launches() - n0) // reps
    clocks = sampler.stop(t0, t1) if sampler else None
    path = g.sweep_path() + ("+jit" if g.last_sweep_specialized() else "")
    g.destroy()
    flips = steps * k * L * L
    ms = float(np.median(events))
    return {"ms": ms, "ms_min": float(min(events)), "ms_max": float(max(events)), "reps": reps, "gpu_seconds": total,
            "flips_per_ns": flips / (ms * 1e6), "launches": int(launches), "path": path, "clocks": clocks}


def time_e2e(P, torch, L, layout, tile, k, steps, rng="planes", packed=False):
    """Same metric through the public API with HOST buffers: every step uploads the spins from
    pinned host memory (ising_set_spins), runs one pass, and reads them back (ising_copy_spins).
    packed: the one-bit-per-site host format (ising_set_spins_bits / ising_copy_spins_bits)."""
    g = P.Ising(2, L, seed=3, rng=rng)
    g.set_jit(JIT)
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    if packed:
        host = torch.empty(L * L // 32, dtype=torch.int32).pin_memory()
        g.copy_spins_bits(host)
        g.set_spins, g.copy_spins = g.set_spins_bits, g.copy_spins_bits
    else:
        host = torch.empty(L * L, dtype=torch.int8).pin_memory()
        g.copy_spins(host)
    g.sweep(W.BETA_C_2D, 1, tile, k)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        g.set_spins(host)
        g.sweep(W.BETA_C_2D, 1, tile, k)
        g.copy_spins(host)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    g.destroy()
    nbytes = host.numel() * host.element_size()
    return {"value": steps * k * L * L / (ms * 1e6), "unit": UNIT, "h2d_bytes_per_step": nbytes,
            "d2h_bytes_per_step": nbytes, "steps": steps,
            "host_format": "one bit per site (ising_set_spins_bits / ising_copy_spins_bits)" if packed else "int8 +-1 (ising_set_spins / ising_copy_spins)"}


def run_config(P, torch, a) -> None:
    """Device-timed flips/ns of another BASELINE.json config (1, 2, 4, 5; config 3 is the default run), planes
    mapping, int8 records unless --layout bits.  One JSON line per (k or beta) variant of the config."""
    c = W.CONFIGS[a.config]
    dim, L = c["dim"], c["L"]
    seeds = list(c.get("seeds", [c.get("seed")]))
    J = W.couplings(dim, L, c["jseed"]) if "jseed" in c else None
    variants = [(c["beta"], k) for k in c.get("ks", [c.get("k")])] if "beta" in c else [(b, c["k"]) for b in c["betas"]]
    for beta, k in variants:
        g = P.Ising(dim, L, coupling=J, seeds=seeds, rng=a.rng)
        g.set_jit(JIT)
        if a.layout == "bits":
            g.set_layout(P.ISING_LAYOUT_BITS)
        n = max(4, min(c["n"], a.steps if a.steps != 50 else c["n"], int(4e10 / (k * len(seeds) * L ** dim))))
        g.sweep(beta, max(a.warmup, min(n, -(-(1 << 27) // (k * len(seeds) * L ** dim)))), c["tile"], k)   # warm-up also compiles
        g.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n0 = P.ising_kernel_launches()
        e0.record()
        g.sweep(beta, n, c["tile"], k)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        flips = n * k * len(seeds) * L ** dim
        # the config's declared outputs, timed apart from the sweeps (the paper excludes measurements from flip times)
        e2, e3, e4 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        Ed = torch.zeros(len(seeds), dtype=torch.int64, device="cuda"); Md = torch.zeros_like(Ed)
        Qd = torch.zeros((len(seeds), len(seeds)), dtype=torch.int64, device="cuda")
        from paper_1006_3865_b200 import binding as Bn
        lib_E = lambda: Bn._check(P.lib().ising_observables(g._h, Bn._ptr(Ed), Bn._ptr(Md)))
        lib_E(); g.overlap_all(Qd); torch.cuda.synchronize()
        e2.record(); lib_E(); e3.record(); g.overlap_all(Qd); e4.record(); torch.cuda.synchronize()
        outputs = {"observables_ms": e2.elapsed_time(e3), "overlap_all_ms": e3.elapsed_time(e4), "pairs": len(seeds) * (len(seeds) - 1) // 2,
                   "whole_job_ms": ms + e2.elapsed_time(e4),
                   "note": f"{n} passes + E, M of every replica + all pairwise overlaps at the end (device buffers)"}
        print(json.dumps({"metric": f"spin flips/ns (BASELINE config {a.config})", "value": flips / (ms * 1e6), "unit": UNIT, "outputs": outputs,
                          "n_gpus": 1, "steps": n, "ms_per_step": ms / n, "higher_is_better": True, "dtype": "u8" if a.layout == "int8" else "u32 bit-planes",
                          "data": "synthetic", "gpu_launches": int(P.ising_kernel_launches() - n0),
                          "config": {"workload": f"BASELINE config {a.config}: dim={dim} L={L} replicas={len(seeds)} J={'+-1 (jseed %d)' % c['jseed'] if J is not None else '+1'} "
                                                 f"beta={beta} tile={c['tile']} k={k} layout={a.layout} rng={a.rng}",
                                     "kernel_path": g.sweep_path() + ("+jit" if g.last_sweep_specialized() else "")}}), flush=True)
        g.destroy()


def run_amsc(P, torch, a) -> None:
    """asynchronous multi-spin coding ("0.15 ps per spin flip").  32 disorder realisations of the
    +-J model per machine word (64: two word lattices), one random number per site; attempted flips per ns summed over the realisations; 2D, and the 3D
    Edwards-Anderson glass."""
    rows = []
    single = a.L != 16384                      # --L given: one variant (--dim, --L, --tile, --k), e.g. for an ncu capture
    cases = [(a.dim, a.L, a.tile, a.k, 32)] if single else \
        [(2, L, T, k, R) for L in (1024, 4096) for T in (32, 64) for k in (1, 4, 16) for R in (32, 64)] + \
        [(3, L, 8, k, R) for L in (64, 128) for k in (1, 4, 16) for R in (32, 64)]
    for dim, L, T, k, R in cases:
        J = W.realisations(dim, L, R, 5)
        g = P.Ising(dim, L, coupling=J, seeds=list(range(100, 100 + R)), sweep_seed=77)
        n = max(4, min(400, int(4e11 / (k * R * L ** dim))))
        g.sweep(1.0, 3, T, k)
        g.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        g.sweep(1.0, n, T, k)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        rows.append({"dim": dim, "L": L, "tile": T, "k": k, "realisations": R, "passes": n, "path": g.sweep_path(),
                     "flips_per_ns": round(n * k * R * L ** dim / (ms * 1e6), 1),
                     "ps_per_flip": round(ms * 1e9 / (n * k * R * L ** dim), 4)})
        g.destroy()
        del J
    print(json.dumps({"study": "amsc", "beta": 1.0, "unit": UNIT, "rows": rows}), flush=True)


def heis_alu_peak(dim: int, sm_mhz: float = 1965.0) -> dict:
    """Issue ceiling of one Heisenberg update on B200: the operations H2-H6 state, costed with the
    pipe rates measured in profiles/r02_microbench.md.  Per warp-update, in SMSP-cycles: half a Philox4x32-10 call
    (109 measured per call, profiles/r02_microbench.md; one call serves two updates), every stated float / convert / bit-field / select operation
    and every shared-memory access one issue slot."""
    fp = 35 + (3 + 6 * (dim - 1)) + 3 + 3 + 3 + 16 + 3       # direction, field adds, d, e, u, P(beta*e), decision
    lsu = 3 * (2 * dim + 1) + 3                              # neighbour + own loads, store of an accepted spin
    cycles = 109.0 / 2 + fp + lsu
    return {"cycles_per_warp_update": cycles, "peak": 148 * 4 * sm_mhz * 1e6 / cycles * 32 / 1e9}


def run_heisenberg(P, torch, a) -> None:
    """the continuous-spin (classical Heisenberg) sweep of P:100 in single precision, include/heisenberg.h.
    Spin updates per ns, device-timed; lattices larger than L2 (three float planes: 805 MB at 2D L=8192, 201 MB at 3D
    L=256).  One JSON line per (dim, L, tile, k); the first carries the CPU oracle timed on a small lattice."""
    single = a.L != 16384
    variants = [(a.dim, a.L, a.tile, a.k)] if single else \
        [(2, 8192, 32, 1), (2, 8192, 32, 4), (2, 8192, 32, 16), (2, 8192, 64, 1), (2, 8192, 64, 4), (2, 8192, 64, 16),
         (3, 256, 8, 1), (3, 256, 8, 4), (3, 256, 8, 16), (3, 256, 16, 4)]
    hbm_gbs, _, sm_mhz = measured_peaks()
    first = True
    for dim, L, T, k in variants:
        beta = 0.7 if dim == 2 else 0.693            # 3D: near the critical coupling 0.6930 of the model
        g = P.Heisenberg(dim, L, seed=3)
        n = max(4, min(a.steps, int(6e9 / (k * L ** dim))))
        g.sweep(beta, max(3, a.warmup), T, k)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n0 = P.ising_kernel_launches()
        e0.record()
        g.sweep(beta, n, T, k)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        upd = n * k * L ** dim / (ms * 1e6)
        alu = heis_alu_peak(dim, sm_mhz)
        bytes_per_update = (12.0 * (1 + 2 * dim / T) + 12.0) / k
        line = {"metric": "spin updates/ns (Heisenberg, single precision)", "value": upd, "unit": "updates/ns", "n_gpus": 1,
                "steps": n, "warmup": max(3, a.warmup), "ms_per_step": ms / n, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic", "gpu_launches": int(P.ising_kernel_launches() - n0),
                "config": {"workload": f"Heisenberg dim={dim} L={L} seed=3 beta={beta} tile={T} k={k}; {3 * 4 * L ** dim / 1e6:.0f} MB of spins (> L2)",
                           "kernel_path": g.sweep_path()},
                "roofline": ({"bound": "alu", "achieved": upd, "peak": alu["peak"], "unit": "updates/ns", "frac": upd / alu["peak"]}
                             if alu["peak"] * bytes_per_update < hbm_gbs else
                             {"bound": "hbm", "achieved": upd * bytes_per_update, "peak": hbm_gbs, "unit": "GB/s",
                              "frac": upd * bytes_per_update / hbm_gbs})}
        line["roofline"].update({"traffic": None, "alu_peak_updates_per_ns": alu["peak"], "alu_frac": upd / alu["peak"],
                                 "cycles_per_warp_update": alu["cycles_per_warp_update"], "bytes_per_update": bytes_per_update,
                                 "hbm_algorithmic_gbs": upd * bytes_per_update, "hbm_frac": upd * bytes_per_update / hbm_gbs,
                                 "note": "bound = the lower of the HBM roofline (algorithmic bytes) and the issue ceiling of the stated operations (DESIGN.md 7.4)"})
        g.destroy()
        if first and not a.no_extras:
            from oracle import heisenberg as HO
            Lo = 256 if dim == 2 else 40
            o = HO.HeisenbergOracle(dim, Lo, seed=3)
            o.sweep(beta, 1, T if Lo % (2 * T) == 0 else 0, 1)
            t0 = time.perf_counter()
            passes = 0
            while time.perf_counter() - t0 < 10.0:
                o.sweep(beta, 4, T if Lo % (2 * T) == 0 else 0, k)
                passes += 4
            dt = time.perf_counter() - t0
            line["cpu_baseline"] = {"value": passes * k * Lo ** dim / (dt * 1e9), "unit": "updates/ns", "cores": 1, "kind": "oracle",
                                    "sample": f"{passes} passes of dim={dim} L={Lo} tile={T} k={k} (same update rule, smaller lattice)"}
        first = False
        print(json.dumps(line), flush=True)


def run_lscan(P, torch, a) -> None:
    """flips/ns against L in the style of the paper's Fig. 3 and its tile tuning, planes mapping, int8
    records: tiles 32 and 64 (the native register tiles) at k = 1, 4, 16; tiles 8, 16, 128 (masked half-sweeps) and the plain
    checkerboard (tile 0 = L) at k = 1."""
    rows = []
    for L in (64, 128, 256, 512, 1024, 2048, 4096, 8192, 16384):
        for T in (8, 16, 32, 64, 128, 0):
            if T and (L % T or (L // T) % 2):
                continue
            for k in ((1, 4, 16) if T in (32, 64) else (1,)):
                n = max(4, min(2000, int(2e10 / (k * L * L))))
                if T not in (32, 64):
                    n = max(4, n // 4)
                r = time_variant(P, torch, L, "int8", T, k, n, 3, None, "planes")
                rows.append({"L": L, "tile": T, "k": k, "passes": n, "flips_per_ns": round(r["flips_per_ns"], 2),
                             "us_per_pass": round(1e3 * r["ms"] / n, 2), "path": r["path"]})
    print(json.dumps({"study": "lscan", "unit": UNIT, "rows": rows}), flush=True)


def run_autocorr(P, torch, a) -> None:
    """what multi-hit costs in autocorrelation.  L=128 at beta_c, tile 32, 4e5 passes after
    2e4 of thermalisation; tau_int of E and |M| in outer passes; independent samples per second of GPU time."""
    from paper_1006_3865_b200.analysis import independent_samples_per_second, tau_int
    L, T, n = 128, 32, 400000
    rows = []
    for k in (1, 2, 4, 8, 16):
        g = P.Ising(2, L, seed=11)
        g.sweep(W.BETA_C_2D, 20000, T, k)
        E = torch.zeros(n, dtype=torch.int64, device="cuda")
        M = torch.zeros(n, dtype=torch.int64, device="cuda")
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        g.sweep_series(W.BETA_C_2D, n, T, k, E=E, M=M)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        tE, _ = tau_int(E.cpu().numpy())
        tM, _ = tau_int(np.abs(M.cpu().numpy()))
        rows.append({"k": k, "tau_E_passes": round(tE, 2), "tau_absM_passes": round(tM, 2),
                     "tau_absM_inner_sweeps": round(tM * k, 2), "seconds": round(dt, 2),
                     "indep_samples_per_s_absM": round(independent_samples_per_second(n, dt, tM), 1)})
        g.destroy()
    print(json.dumps({"study": "autocorr", "L": L, "tile": T, "beta": W.BETA_C_2D, "passes": n, "rows": rows}), flush=True)


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--layout", default="int8", choices=["int8", "bits"])
    ap.add_argument("--tile", type=int, default=64)
    ap.add_argument("--k", type=int, default=1)
    ap.add_argument("--rng", default="planes", choices=["planes", "words"], help="RNG->site mapping (DESIGN.md R6)")
    ap.add_argument("--L", type=int, default=16384)
    ap.add_argument("--min-seconds", type=float, default=1.0,
                    help="repeat the timed K-step call back to back until this much GPU time has elapsed; value = median repetition")
    ap.add_argument("--no-extras", action="store_true", help="skip e2e, cpu_baseline and the k/tile table")
    ap.add_argument("--jit", default="auto", choices=["auto", "on", "off"], help="run-time kernel specialisation (ising_set_jit)")
    ap.add_argument("--force-path", type=int, default=0, choices=[0, 2, 3, 4],
                    help="ising_force_path: 2 = a launch per coarse colour, 3 = no data-flow kernel, 4 = no on-chip (cluster / grid) kernels")
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5], help="time another BASELINE config (default 3 = the headline run)")
    ap.add_argument("--amsc", action="store_true", help="study: asynchronous multi-spin coding throughput (SURVEY 8(f)-1)")
    ap.add_argument("--heisenberg", action="store_true", help="study: the continuous-spin (Heisenberg) sweep, include/heisenberg.h (SURVEY 8(f)-4)")
    ap.add_argument("--dim", type=int, default=2, choices=[2, 3], help="with --heisenberg --L: lattice dimension")
    ap.add_argument("--lscan", action="store_true", help="study: flips/ns against L (SURVEY 8(f)-3)")
    ap.add_argument("--autocorr", action="store_true", help="study: autocorrelation time against k (SURVEY 8(f)-2)")
    ap.add_argument("--selftest-ranks", action="store_true", help="CPU/gloo check of the multi-rank aggregation, no GPU")
    a = ap.parse_args()
    global JIT, FORCE
    JIT = a.jit
    FORCE = a.force_path
    a.warmup = max(a.warmup, 3) if a.impl == "ours" else a.warmup
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if a.selftest_ranks:
        selftest_ranks(rank, world)
        return
    if a.impl == "reference":
        run_reference(a, rank, world)
        return

    import torch
    import paper_1006_3865_b200 as P
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the product has no CPU path")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    P.use_torch()
    L = a.L
    if a.lscan or a.autocorr or a.amsc or a.heisenberg:
        (run_lscan if a.lscan else run_autocorr if a.autocorr else run_amsc if a.amsc else run_heisenberg)(P, torch, a)
        return
    if a.config != 3:
        run_config(P, torch, a)
        return

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    res = time_variant(P, torch, L, a.layout, a.tile, a.k, a.steps, a.warmup, sampler, a.rng, min_seconds=a.min_seconds, max_reps=2000)
    barrier()
    ms, value = aggregate_replicas(res["ms"], world, a.steps, a.k, L, dist, "cuda")

    peak, peak_src, sm_max = measured_peaks()
    family = ("flow" if res["path"].startswith("flow") else "tile" if res["path"].startswith("tile_planes") else
              "grid" if res["path"].startswith("grid_planes") else res["path"])
    ncu = NCU.get((a.rng, a.layout, a.tile, a.k, family)) if L == 16384 and res["path"].endswith("+jit") else None
    ncu_stale = ncu is not None and kernel_fingerprint(family) != ncu["fp"]
    if ncu_stale:            # the kernel changed since the capture: quote nothing from it
        ncu = None
    traffic, warp_instr = ncu_per_phase(ncu, a.steps)
    bpf = algorithmic_bytes_per_flip(a.tile, a.k, a.layout, L)
    launches_per_step = 2
    bytes_per_launch = bpf * a.k * L * L / launches_per_step
    launch_ms = res["ms"] / (a.steps * launches_per_step)
    achieved = bytes_per_launch / (launch_ms * 1e6)            # GB/s
    lat_bytes = L * L if a.layout == "int8" else L * L // 8
    on_chip = res["path"].startswith("grid_")          # k_grid_planes, and k_grid_plain for the plain / masked schemes
    hbm = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
           "frac_of_8TBs_nominal": achieved / 8000.0, "algorithmic_bytes_per_flip": bpf}
    issue = ({"bound": "alu", "unit": "G warp-instr/s", "achieved": warp_instr / (launch_ms * 1e6),
              "peak": issue_peak_gips(sm_max), "frac": warp_instr / (launch_ms * 1e6) / issue_peak_gips(sm_max),
              "peak_source": "148 SMs x 4 schedulers x one warp-instruction per cycle x sm_max_mhz (DESIGN.md 7.3)",
              "kind": "issue slots (one warp-instruction per scheduler cycle, 592 schedulers)",
              "warp_instr_per_phase": warp_instr,
              "note": "what binds is not the slot count but the dispatch model of DESIGN.md 7.3 / profiles/r02_microbench.md "
                      "(a 16-lane ALU instruction holds the scheduler 2 cycles, a wide multiply 2.25): a model, not a hardware counter"}
             if warp_instr else None)
    common = {"traffic": traffic,
              "traffic_source": ("ncu dram__bytes_read.sum + dram__bytes_write.sum per phase, " + ncu.get("source", "profiles/")) if ncu else None,
              "traffic_stale": ncu_stale, "kernel": f"{res['path']}<{a.tile}>", "avg_launch_ms": launch_ms}
    if on_chip:
        # The lattice stays in shared memory for the whole call: DRAM sees it once per call, not once per phase, and the
        # kernel is bound by instruction issue.  The roofline is therefore the ALU one; the algorithmic-bytes figure of
        # SURVEY 8(d) (what a kernel that streams the lattice every pass must move) is kept beside it for comparison.
        roof = dict(issue) if issue else {"bound": "alu", "unit": "G warp-instr/s", "achieved": None, "peak": issue_peak_gips(sm_max), "frac": None}
        roof.update(common)
        if ncu and "pipes_16_passes" in ncu:        # hardware counters of the committed 16-pass capture (not of this run)
            roof["ncu_pipe_utilisation"] = dict(ncu["pipes_16_passes"], source=ncu["source"] + ": sm__pipe_alu_cycles_active, "
                                                "sm__pipe_fmaheavy_cycles_active, sm__issue_active (.avg.pct_of_peak_sustained_elapsed / 100)")
        roof["launch_unit"] = ("one phase (coarse colour of a pass) of the cooperative launch that keeps the lattice on chip: CUDA-event time "
                               "of the call / (2 * steps), the load and the store of the lattice (once per call) included")
        roof["hbm_algorithmic"] = dict(hbm, note="bytes a kernel that streams the lattice every pass would move (SURVEY 8(d)) / measured time: "
                                                 f"such a kernel cannot exceed {peak / bpf:.0f} flips/ns; this one moves traffic / algorithmic "
                                                 "of them (the lattice crosses HBM once per call)")
    else:
        roof = dict(hbm)
        roof.update(common)
        roof["launch_unit"] = ("one launch of k_tile_planes = one coarse colour of one pass" if res["path"].startswith("tile") else
                               "one phase (coarse colour of a pass) of the persistent launch: CUDA-event time of the call / (2 * steps)")
        roof["issue"] = issue
    how = ("(2 launches)" if res["path"].startswith("tile") else
           "(all steps of a call in one cooperative launch, the lattice in shared memory from the first pass to the last)" if on_chip else
           "(all steps of a call in one persistent launch)")
    line = {"metric": METRIC if L == 16384 else f"spin flips/ns (2D Ising L={L}, beta_c)", "value": value, "unit": UNIT,
            "n_gpus": world, "steps": a.steps, "warmup": a.warmup,
            "ms_per_step": ms / a.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "u8" if a.layout == "int8" else "u32 bit-planes", "data": "synthetic",
            "config": {"workload": f"{'BASELINE config 3' if L == 16384 else 'config 3 at another size'}: 2D Ising L={L} hot start seed 3 "
                                   f"beta=0.4406868 layout={a.layout} rng={a.rng} tile={a.tile} k={a.k}; one step = one outer pass " + how,
                       "l2": (f"lattice ({lat_bytes / 2 ** 20:g} MiB {a.layout}) exceeds the 126 MB L2; no explicit flush" if lat_bytes > 126e6
                              else f"lattice ({lat_bytes / 2 ** 20:g} MiB {a.layout}) fits L2: not an HBM claim")
                             + ("; on chip between the passes of a call: read from and written to HBM once per call, inside the timed region" if on_chip else ""),
                       "kernel_path": res["path"], "parallelism": "replicas only" if world > 1 else "single GPU"},
            "ns_per_flip": 1.0 / value, "gpu_launches": res["launches"], "clocks": res["clocks"],
            "repetitions": {"n": res["reps"], "each": f"one ising_sweep({a.steps}) call = exactly {a.steps} steps, CUDA events around it",
                            "reported": "median", "gpu_seconds": res["gpu_seconds"],
                            "value_min": a.steps * a.k * L * L / (res["ms_max"] * 1e6) * world,
                            "value_max": a.steps * a.k * L * L / (res["ms_min"] * 1e6) * world},
            "roofline": roof}
    if rank == 0 and not a.no_extras and world == 1:
        table = {}
        for rng, lay in (("planes", "int8"), ("planes", "bits"), ("words", "int8")):
            for T in (32, 64):
                for k in (1, 4, 16):
                    st = max(2, min(a.steps, 40 // k))
                    r = time_variant(P, torch, L, lay, T, k, st, 3, None, rng, min_seconds=0.25, max_reps=400)
                    table[f"{rng}_{lay}_t{T}_k{k}"] = {"flips_per_ns": round(r["flips_per_ns"], 1), "steps": st, "reps": r["reps"], "kernel_path": r["path"],
                                                "hbm_GBs": round(r["flips_per_ns"] * algorithmic_bytes_per_flip(T, k, lay), 1)}
        # the headline variant through the kernels that stream the lattice through HBM every pass (ising_force_path 4: the
        # persistent data-flow kernel; 2: a launch per coarse colour): the HBM-bound forms of the same call
        for T in (64, 32):
            for fp, name in ((4, "flow"), (2, "launches")):
                st = max(2, min(a.steps, 40))
                r = time_variant(P, torch, L, "int8", T, 1, st, 3, None, "planes", min_seconds=0.25, max_reps=400, force=fp)
                table[f"planes_int8_t{T}_k1_hbm_{name}"] = {"flips_per_ns": round(r["flips_per_ns"], 1), "steps": st, "reps": r["reps"], "kernel_path": r["path"],
                                                           "hbm_GBs": round(r["flips_per_ns"] * algorithmic_bytes_per_flip(T, 1, "int8"), 1),
                                                           "hbm_frac": round(r["flips_per_ns"] * algorithmic_bytes_per_flip(T, 1, "int8") / peak, 3)}
        # the scheme the paper starts from (row a8): plain checkerboard, tile == L, a launch per half-sweep
        for lay in ("int8", "bits"):
            st = max(2, min(a.steps, 40))
            r = time_variant(P, torch, L, lay, L, 1, st, 3, None, "planes", min_seconds=0.25, max_reps=400)
            table[f"planes_{lay}_plain"] = {"flips_per_ns": round(r["flips_per_ns"], 1), "steps": st, "kernel_path": r["path"],
                                            "hbm_GBs": round(r["flips_per_ns"] * algorithmic_bytes_per_flip(L, 1, lay, L), 1)}
        line["variants"] = table
        line["e2e"] = time_e2e(P, torch, L, a.layout, a.tile, a.k, 3, a.rng)
        line["e2e_bits"] = time_e2e(P, torch, L, a.layout, a.tile, a.k, 3, a.rng, packed=True)
        ncores = 1
        v, dt = oracle_flips_per_ns(L, a.tile, a.k, 2, a.rng)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": ncores, "kind": "oracle",
                                "sample": f"2 outer passes of the full L={L} lattice (tile {a.tile}, k {a.k}), {dt:.1f} s, "
                                          f"host has {os.cpu_count()} cores, oracle is sequential"}
    elif rank == 0:
        line["e2e"] = None
    if rank == 0:
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
