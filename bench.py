#!/usr/bin/env python
"""bench.py -- R-matrix formation throughput on B200 (eq. 4 of arxiv 1909.07321).

A "step" is one pass of the whole hot path (pole scaling, TMA staging, DMMA SYRK, mirrored
store, scheduler: SURVEY.md 8a S1-S5) over one synthetic workload, through the C ABI of
libpstgf_rmat.so.  Default workload: BASELINE.json configs[4], the "large single partial wave"
the north_star's >= 70 % target is quoted on (n_chan 512, n_poles 10240, n_E 256); --config 1..5
selects another (2-5 are parity-test sizes as well).

    python bench.py --gpus 1 --steps 10 --warmup 3            # this repo's CUDA path
    python bench.py --impl reference --steps 3 --warmup 1     # the CPU oracle as it stands

One JSON line on stdout (rank 0).  See DESIGN.md "Measurement" for every key.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "R-matrix energies/s"
UNIT = "energies/s"
# FP64 nominal ratio used when the DMMA probe is not run: FP64 tensor 45 TFLOP/s per B200
# (/opt/skills/guides/blackwell_cuda_programming.md:52) over bf16 dense 2250 TFLOP/s (B200_PROFILING.md:36).
FP64_OVER_BF16_NOMINAL = 45.0 / 2250.0
FALLBACK_BF16_TFLOPS = 1590.0      # B200_PROFILING.md fallback, used only if MEASURED_PEAKS.json is absent
FALLBACK_HBM_GBS = 6650.0
PAPER_ENERGIES_PER_S = 1.0 / 14.0  # "14-18 secs per R-matrix formation" at 7261 channels x 106 661 poles


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["cuda", "reference"], default="cuda")
    ap.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5, 6, 7],
                    help="1-5: BASELINE.json configs[0..4]; 6: the paper-scale wave of PAPER.md:168 (7261 x 106661); "
                         "7: 256 small waves, n_chan in [8, 32] (PAPER.md:676 shape: many partial waves in one call)")
    ap.add_argument("--n-E", type=int, default=0, dest="n_E",
                    help="override the energies per wave (the mesh keeps its range): PSTGF calls RINIT once per "
                         "(wave, energy), PAPER.md:122-126, so few-energy calls are a workload of their own")
    ap.add_argument("--w-layout", choices=["poles", "channels"], default="poles",
                    help="memory order of W on the device: pole-contiguous [n_chan][n_poles] (default, north_star's) or "
                         "channel-contiguous [n_poles][n_chan], the H.DAT record order of PAPER.md:535")
    ap.add_argument("--prior-art", action="store_true",
                    help="also time the paper's own GPU scheme (PAPER.md:164-166: scaled copy, 10 upper-triangle block "
                         "multiplies per energy, symmetrise) with cuBLAS DGEMM through torch.matmul: context, not a path "
                         "of the library")
    ap.add_argument("--tail-policy", choices=["auto", "none", "all"], default="auto",
                    help="scheduling knob of the library (pstgf_rmat_set_tail_policy): fine-tile tail sized automatically "
                         "(default), coarse tiles only, fine tiles only; same bits, for measurements")
    ap.add_argument("--slab-policy", choices=["auto", "none", "32", "64", "128"], default="auto",
                    help="how the n_E mod 8 energies are cut (pstgf_debug_set_slab_policy): tile edge chosen by the planner "
                         "(default), left to a partly idle block of 8 (round-1 behaviour), or a forced edge; same bits")
    ap.add_argument("--e2e-chunk-mib", type=int, default=0,
                    help="max_chunk_bytes of pstgf_rmat_form_batch_host in MiB (0 = the library's default)")
    ap.add_argument("--scaling", choices=["weak", "strong"], default="weak",
                    help="N > 1 ranks: weak = the configuration with an N times finer mesh (per-rank work fixed, default); "
                         "strong = the configuration as it is, its energy blocks split over the ranks (total work fixed)")
    ap.add_argument("--variant", choices=["dmma", "sliced"], default="dmma",
                    help="dmma: the library's path (default).  sliced: pstgf_rmat_form_sliced, the INT8 tcgen05 VARIANT of "
                         "SURVEY.md 8f-4 (single-wave configs only; results agree with FP64 sums to ~1e-12, see the header); "
                         "a comparison line, not the product's number")
    ap.add_argument("--slices", type=int, default=7, help="digits per element for --variant sliced (7: ~1e-12, 8: ~1e-14)")
    ap.add_argument("--probe-i8", action="store_true",
                    help="also run the INT8 tensor-pipe probe (tcgen05.mma kind::i8, measure/i8_probe.cu) and report its rate "
                         "under context.int8_tensor_pops: the number behind DESIGN.md 11.6, not a path of the library")
    ap.add_argument("--probe-l2", action="store_true",
                    help="run ONLY the L2 -> shared-memory load-rate probe (measure/l2_probe.cu: TMA boxes of several inner "
                         "extents, 1-D bulk copies, issuing lanes, ring depths, multicast over 2 and 4 CTAs) and print its table")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing leg")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end leg")
    ap.add_argument("--no-all-configs", action="store_true",
                    help="skip the `all_configs` entries (configs 1-4 and n_E = 1 / 32 on config 5's wave, 5 steps each) "
                         "that the default config-5 run adds to its line")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target CPU time of the oracle sample")
    return ap.parse_args()


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return dict(source="measured", hbm_gbs=float(p["hbm_gbs"]), bf16=float(p["bf16_tflops"]),
                    bf16_sustained=float(p.get("bf16_tflops_sustained", p["bf16_tflops"])),
                    sm_max_mhz=float(p.get("sm_max_mhz", 1965.0)))
    return dict(source="fallback", hbm_gbs=FALLBACK_HBM_GBS, bf16=FALLBACK_BF16_TFLOPS, bf16_sustained=1400.0,
                sm_max_mhz=1965.0)


# ---- clocks ----------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi -lms sampling of SM clock and throttle reasons during the timed region."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.file = None

    def start(self):
        try:
            self.file = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits",
                                          "-lms", "50", "-i", str(self.index)], stdout=self.file, stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.file.flush()
        self.file.seek(0)
        clocks, reasons, power, cmax = [], set(), [], None
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.file.read().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                clocks.append(float(parts[0]))
                cmax = float(parts[1])
                power.append(float(parts[2]))
            except ValueError:
                continue
            for nm, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.file.close()
        try:
            os.unlink(self.file.name)
        except OSError:
            pass
        if clocks:
            clocks.sort()
            out.update(sm_mhz=clocks[len(clocks) // 2], sm_max_mhz=cmax, reasons=sorted(reasons), samples=len(clocks),
                       power_w_max=max(power) if power else None)
        return out


# ---- workload --------------------------------------------------------------------------------
def job_workload(args, world: int):
    """The workload of the whole job (all ranks): the configuration as it is at N = 1 and under --scaling strong,
    the configuration with an N times finer mesh under --scaling weak (per-rank work fixed)."""
    from paper_1909_07321_b200 import inputs
    if world == 1 or args.scaling == "strong":
        return inputs.make_config(args.config, n_E=args.n_E or None)
    base = inputs.config_shapes(args.config)
    return inputs.make_config(args.config, n_E=world * (args.n_E or base[0][2]))


def rank_workload(wl_job, rank: int, world: int):
    """This rank's share of the job: shard.plan's wave-rotated sets of energy blocks (Fig. 1),
    waves in the rank's visiting order.  The whole job at world == 1."""
    import numpy as np
    from paper_1909_07321_b200 import inputs, shard
    if world == 1:
        return wl_job
    wl = inputs.Workload(name=wl_job.name, seed=wl_job.seed)
    for p, idx in shard.plan([w.n_E for w in wl_job.waves], rank, world):
        w = wl_job.waves[p]
        wl.waves.append(inputs.Wave(w.W, w.E_k, np.ascontiguousarray(w.energies[idx]), w.a))
    return wl


def workload_description(cfg: int, wl) -> dict:
    names = {1: "configs[0] single wave 8x160, n_E 1000", 2: "configs[1] single wave 64x1280, n_E 4096",
             3: "configs[2] 8 waves 256x5120, n_E 2048 shared", 4: "configs[3] ragged 32 waves n_chan U[16,400], n_E 512",
             5: "configs[4] large single wave 512x10240, n_E 256",
             6: "paper-scale single wave 7261x106661 (PAPER.md:168), n_E 16 [not in BASELINE.json configs]",
             7: "256 small waves n_chan U[8,32], n_poles 20 n_chan, n_E 512 [not in BASELINE.json configs]"}
    return {"workload": names[cfg], "config_index": cfg - 1, "seed": wl.seed, "n_waves": len(wl.waves),
            "n_chan": [w.n_chan for w in wl.waves] if len(wl.waves) <= 8 else
            {"min": min(w.n_chan for w in wl.waves), "max": max(w.n_chan for w in wl.waves)},
            "n_energies_per_step": wl.n_energies(), "counted_flop_per_step": wl.counted_flop(),
            "r_bytes_per_step": wl.r_bytes(), "parallelism": "energy blocks sharded over ranks, wave-rotated (shard.plan); no collective"}


# ---- CPU oracle legs (the only places bench.py touches oracle/) ---------------------------------
def oracle_sample_run(wl, energies_per_wave: int, threads: int):
    """Time the oracle, as it stands, on the first `energies_per_wave` energies of every wave."""
    from oracle import rmat_oracle
    t0 = time.perf_counter()
    n = 0
    for w in wl.waves:
        k = min(energies_per_wave, w.n_E)
        rmat_oracle.rmat_form(w.W, w.E_k, w.energies[:k], w.a, threads=threads)
        n += k
    return n, time.perf_counter() - t0


def oracle_cores():
    from oracle import rmat_oracle
    rmat_oracle.build()
    return max(1, min(rmat_oracle.max_threads(), os.cpu_count() or 1))


def est_oracle_seconds_per_energy(wl) -> float:
    # ~2.6 ns per compensated term (SURVEY.md 8d probe), C(C+1)/2 * K terms... the oracle fills all C^2 entries
    return sum(2.6e-9 * w.n_chan * w.n_chan * w.n_poles for w in wl.waves) / max(1, len(wl.waves))


def cpu_baseline_entries(wl, target_seconds: float, cores: int) -> dict:
    """Waves whose single energy would take the oracle hours (config 6): time it on seeded sampled entries.
    Every entry of a wave costs the same n_poles terms, so energies/s = entries/s / n_chan^2 exactly."""
    import numpy as np
    from oracle import rmat_oracle
    w = wl.waves[0]
    S = int(max(cores, target_seconds * cores / (2.6e-9 * w.n_poles)))
    rng = np.random.default_rng(7)
    e_idx, n_idx, m_idx = rng.integers(0, w.n_E, S), rng.integers(0, w.n_chan, S), rng.integers(0, w.n_chan, S)
    t0 = time.perf_counter()
    rmat_oracle.rmat_entries(w.W, w.E_k, w.energies, w.a, e_idx, n_idx, m_idx, threads=cores)
    dt = time.perf_counter() - t0
    return {"value": S / dt / (w.n_chan ** 2), "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{S} seeded entries R[e][n][m] of the wave ({dt:.2f} s wall, OpenMP over entries); one dense "
                      f"energy is {w.n_chan ** 2} entries of equal cost, so energies/s = entries/s / n_chan^2",
            "counted_gflops": S * w.n_poles / dt / 1e9}


def sample_energies_per_wave(wl, seconds: float, cores: int) -> int:
    """Energies per wave for about `seconds` of wall time with `cores` threads over the energies of a wave: a whole
    multiple of the core count (rounded UP, so that no core idles and the oracle is timed at full occupancy), capped
    by the shortest mesh."""
    per_e = est_oracle_seconds_per_energy(wl)                   # one thread, one energy of an average wave
    k = max(1, round(seconds * cores / (per_e * len(wl.waves))))
    k = -(-k // cores) * cores
    return int(min(k, min(w.n_E for w in wl.waves)))


def cpu_baseline(wl, target_seconds: float) -> dict:
    cores = oracle_cores()
    per_e = est_oracle_seconds_per_energy(wl)
    if len(wl.waves) == 1 and per_e > 4 * target_seconds * cores:
        return cpu_baseline_entries(wl, target_seconds, cores)
    k = sample_energies_per_wave(wl, target_seconds, cores)
    n, dt = oracle_sample_run(wl, k, cores)
    # the same loop on ONE thread, on a sample of about a fifth of the CPU time
    k1 = int(max(1, min(min(w.n_E for w in wl.waves), round(0.2 * target_seconds / (per_e * len(wl.waves))))))
    n1, dt1 = oracle_sample_run(wl, k1, 1)
    return {"value": n / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"first {k} energies of each of {len(wl.waves)} wave(s), {n} energies, {dt:.2f} s wall, "
                      f"OpenMP over energies; every energy of a wave costs the same, so energies/s extrapolates",
            "counted_gflops": n and sum(min(k, w.n_E) * w.n_chan ** 2 * w.n_poles for w in wl.waves) / dt / 1e9,
            "one_thread": {"value": n1 / dt1, "unit": UNIT, "cores": 1,
                           "sample": f"first {k1} energies of each wave, {n1} energies, {dt1:.2f} s wall"}}


def run_reference(args):
    """--impl reference: the oracle on the host cores; each step a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    wl = job_workload(args, int(os.environ.get("WORLD_SIZE", "1")))
    cores = oracle_cores()
    per_e = est_oracle_seconds_per_energy(wl)
    budget = 120.0 / max(1, args.steps + args.warmup)            # whole run within a few minutes
    if len(wl.waves) == 1 and per_e > 4 * budget * cores:        # config 6: sampled entries, see cpu_baseline_entries
        for _ in range(args.warmup):
            cpu_baseline_entries(wl, min(budget, 20.0) / 4, cores)
        runs = [cpu_baseline_entries(wl, min(budget, 20.0), cores) for _ in range(args.steps)]
        value = len(runs) / sum(1.0 / r["value"] for r in runs)
        line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 0, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": None, "higher_is_better": True, "scaling": args.scaling,
                "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": workload_description(args.config, wl),
                "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                                 "sample": "each step: " + runs[0]["sample"]},
                "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
        print(json.dumps(line), flush=True)
        return 0
    k = sample_energies_per_wave(wl, min(budget, 20.0), cores)
    for _ in range(args.warmup):
        oracle_sample_run(wl, k, cores)
    total_n, total_t = 0, 0.0
    for _ in range(args.steps):
        n, dt = oracle_sample_run(wl, k, cores)
        total_n += n
        total_t += dt
    value = total_n / total_t
    sample = f"each step: first {k} energies of each of {len(wl.waves)} wave(s) ({total_n // max(1, args.steps)} energies)"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 0, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * total_t / max(1, args.steps), "higher_is_better": True,
            "scaling": args.scaling, "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_description(args.config, wl),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


def ncu_traffic(cfg: int):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the SYRK kernel from the committed
    `ncu --set full` capture (profiles/traffic.csv: config,dram_bytes_per_launch,...), else None."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(path):
        return None
    with open(path) as f:
        for line in f:
            parts = line.strip().split(",")
            if parts and parts[0] == str(cfg):
                try:
                    return float(parts[1])
                except (ValueError, IndexError):
                    return None
    return None


# ---- prior art on the same GPU (context) ---------------------------------------------------------
def prior_art_leg(wl, n_sample: int = 16, library_R=None) -> dict:
    """The scheme the paper describes for its CUDA-Fortran RINIT (Fig. 2), with a library DGEMM
    (cuBLAS through torch.matmul, float64) standing in for its matrix-multiply routine: per energy, form the scaled
    copy W diag(d), compute the 10 upper-triangle blocks of a 4 x 4 block grid one after another, symmetrise.
    Timed on the first `n_sample` energies of every wave with CUDA events; every energy costs the same.
    library_R: per wave, this library's R for (at least) those energies (host or device tensors): the comparator's
    result is checked against it, so that what is timed is known to be eq. 4 (reported as max_rel_err_vs_library,
    the parity tests' per-energy measure)."""
    import torch
    total_ms, n_done, worst = 0.0, 0, 0.0
    for wi, w in enumerate(wl.waves):
        W = torch.from_numpy(w.W).cuda()
        Ek = torch.from_numpy(w.E_k).cuda()
        en = torch.from_numpy(w.energies).cuda()
        C = w.n_chan
        cuts = [round(i * C / 4) for i in range(5)]
        blocks = [(cuts[i], cuts[i + 1]) for i in range(4) if cuts[i + 1] > cuts[i]]
        k = min(n_sample, w.n_E)
        R = torch.empty((k, C, C), dtype=torch.float64, device="cuda")

        def form(e):
            Ws = W * (1.0 / (Ek - en[e]))                       # the scaled operand, a full copy in HBM
            for bi, (r0, r1) in enumerate(blocks):
                for (c0, c1) in blocks[bi:]:
                    blk = torch.matmul(W[r0:r1], Ws[c0:c1].t())
                    R[e, r0:r1, c0:c1] = blk
                    if c0 != r0:
                        R[e, c0:c1, r0:r1] = blk.t()            # "symmetrised to provide the full result"
            R[e].mul_(1.0 / (2.0 * w.a))

        for e in range(min(3, k)):
            form(e)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for e in range(k):
            form(e)
        e1.record()
        torch.cuda.synchronize()
        total_ms += e0.elapsed_time(e1)
        n_done += k
        if library_R is not None:
            ref = library_R[wi][:k].to("cuda")
            num = (R - ref).abs().reshape(k, -1).amax(1)
            den = ref.abs().reshape(k, -1).amax(1)
            worst = max(worst, float((num / den).max()))
    # a stronger library baseline: scaled copies of 8 energies at once and ONE batched DGEMM for the full squares
    b_ms, b_done = 0.0, 0
    for w in wl.waves:
        W = torch.from_numpy(w.W).cuda()
        Ek = torch.from_numpy(w.E_k).cuda()
        en = torch.from_numpy(w.energies).cuda()
        k = min(n_sample, w.n_E)
        k -= k % 8 if k >= 8 else 0
        Rb = torch.empty((k, w.n_chan, w.n_chan), dtype=torch.float64, device="cuda")

        def form_batched():
            for e in range(0, k, 8):
                d = 1.0 / (Ek[None, :] - en[e:e + 8, None])                    # [8, K]
                torch.matmul(W[None] * d[:, None, :], W.t(), out=Rb[e:e + 8])   # [8, C, K] scaled copies, batched DGEMM
            Rb.mul_(1.0 / (2.0 * w.a))

        form_batched()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        form_batched()
        e1.record()
        torch.cuda.synchronize()
        b_ms += e0.elapsed_time(e1)
        b_done += k
    flop = sum(min(n_sample, w.n_E) * w.n_chan ** 2 * w.n_poles for w in wl.waves)
    return {"cublas_batched": {"value": b_done / (b_ms * 1e-3), "unit": UNIT,
                               "kind": "scaled copies of 8 energies + one batched cuBLAS DGEMM of the full squares (torch.matmul)",
                               "sample": f"{b_done} energies, {b_ms:.2f} ms"},
            "value": n_done / (total_ms * 1e-3), "unit": UNIT, "kind": "paper's scheme (PAPER.md:164-166) with cuBLAS DGEMM via "
            "torch.matmul: scaled copy + 10 upper-triangle block multiplies + symmetrise, one energy at a time",
            "sample": f"first {n_sample} energies of each wave ({n_done} energies, {total_ms:.2f} ms)",
            "tflops_counted": flop / (total_ms * 1e-3) / 1e12,
            "max_rel_err_vs_library": worst if library_R is not None else None}


# ---- the other configurations, in the same line ------------------------------------------------------
def quick_config_line(cfg: int, n_E, peak_tflops: float, flush_buf, device_index: int, steps: int = 5, warmup: int = 3) -> dict:
    """One configuration through the device-pointer calls, timed like the headline (L2 flushed between steps, CUDA
    events on the launch stream, clocks sampled during its own timed region), as an entry of `all_configs`."""
    import torch
    from paper_1909_07321_b200 import inputs, rmat
    wl = inputs.make_config(cfg, n_E=n_E)
    dev, shared = [], {}
    for w in wl.waves:
        key = id(w.energies)
        if key not in shared:
            shared[key] = torch.from_numpy(w.energies).cuda()
        R = torch.empty((w.n_E, w.n_chan, w.n_chan), dtype=torch.float64, device="cuda")
        dev.append((torch.from_numpy(w.W).cuda(), torch.from_numpy(w.E_k).cuda(), shared[key], w.a, R))
    if len(dev) > 1:
        arr = rmat.make_wave_array(dev)
        ws = torch.empty(rmat.pstgf_rmat_batch_workspace_bytes(arr), dtype=torch.uint8, device="cuda")

    def step():
        if len(dev) == 1:
            W, E_k, en, a, R = dev[0]
            rmat.pstgf_rmat_form(W, E_k, en, a, R_out=R)
        else:
            rmat.pstgf_rmat_form_batch(arr, ws)
        return rmat.pstgf_last_launch_count()

    for _ in range(warmup):
        flush_buf.zero_()
        step()
    torch.cuda.synchronize()
    sampler = ClockSampler(device_index)
    sampler.start()
    time.sleep(0.12)
    ms, launches = [], 0
    t_end = time.perf_counter() + 0.25                     # at least a quarter of a second under load for the clock samples
    while len(ms) < steps or time.perf_counter() < t_end:
        flush_buf.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        n = step()
        e1.record()
        torch.cuda.synchronize()
        if len(ms) < steps:
            ms.append(e0.elapsed_time(e1))
            launches += n
    clocks = sampler.stop()
    t = sum(ms) / len(ms)
    tf = wl.counted_flop() / (t * 1e-3) / 1e12
    return {"config": cfg, "n_E": n_E, "workload": workload_description(cfg, wl)["workload"] + (f", n_E overridden to {n_E}" if n_E else ""),
            "steps": len(ms), "warmup": warmup, "ms_per_step": t, "step_ms_min_max": [min(ms), max(ms)],
            "energies_per_s": wl.n_energies() / (t * 1e-3), "tflops_counted": tf, "frac": tf / peak_tflops,
            "gpu_launches": launches, "clocks": clocks}


# ---- L2 -> SM load-rate probe ------------------------------------------------------
def l2_probe_table(device_index: int, sm_mhz: float) -> list:
    """Every row of probe.L2_PROBE_SWEEP on all SMs: best of 3 launches over a 32 MB array (L2-resident after the
    first pass), CUDA events.  delivered = bytes that arrived in shared memory; from_l2 = delivered / cluster size."""
    import torch
    from paper_1909_07321_b200.measure import probe
    sms = torch.cuda.get_device_properties(device_index).multi_processor_count
    src = torch.zeros(400 * probe.L2_PROBE_PITCH, dtype=torch.uint8, device="cuda")
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    rows = []
    for label, mode, inner, box_rows, bps, lanes, stages, cluster in probe.L2_PROBE_SWEEP:
        stage_bytes = inner * box_rows * bps
        iters = max(4 * stages, (64 << 20) // stage_bytes)
        n_ctas = sms - sms % cluster
        best = None
        for rep in range(4):                                  # the first pass loads L2 and the kernel
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            delivered = probe.l2_probe(mode, inner, box_rows, bps, lanes, stages, cluster, iters, n_ctas, src, status)
            e1.record()
            torch.cuda.synchronize()
            if rep:
                best = e0.elapsed_time(e1) if best is None else min(best, e0.elapsed_time(e1))
        if int(status.item()) != 0:
            raise RuntimeError(f"l2 probe timed out in {label!r}")
        tbs = delivered / (best * 1e-3) / 1e12
        rows.append({"pattern": label, "cluster": cluster, "in_flight_kb_per_cta": stages * stage_bytes / 1024,
                     "delivered_tb_s": tbs, "delivered_b_per_clk_per_sm": delivered / (best * 1e-3) / (sm_mhz * 1e6) / n_ctas,
                     "from_l2_tb_s": tbs / cluster, "ms": best})
    return rows


# ---- CUDA arm ----------------------------------------------------------------------------------
def run_cuda(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_1909_07321_b200 import inputs, rmat

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU fallback for the product path")
    torch.cuda.set_device(local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    rmat.load()          # raises if libpstgf_rmat.so is missing
    rmat.pstgf_debug_set_tail_policy({"auto": rmat.PSTGF_TAIL_AUTO, "none": rmat.PSTGF_TAIL_NONE,
                                      "all": rmat.PSTGF_TAIL_ALL}[args.tail_policy])
    rmat.pstgf_debug_set_slab_policy({"auto": rmat.PSTGF_SLAB_AUTO, "none": rmat.PSTGF_SLAB_NONE, "32": rmat.PSTGF_SLAB_T32,
                                      "64": rmat.PSTGF_SLAB_T64, "128": rmat.PSTGF_SLAB_T128}[args.slab_policy])
    peaks = measured_peaks()
    if args.probe_l2:
        if rank == 0:
            sampler = ClockSampler(local_rank)
            sampler.start()
            table = l2_probe_table(local_rank, peaks["sm_max_mhz"])
            print(json.dumps({"probe": "l2_to_shared_memory", "unit": "TB/s delivered into shared memory, all SMs",
                              "source": "32 MB array, L2-resident; one issuing warp per CTA, one CTA per SM, best of 3",
                              "sm_mhz_assumed": peaks["sm_max_mhz"], "rows": table, "clocks": sampler.stop()}), flush=True)
        if world > 1:
            dist.destroy_process_group()
        return 0

    # Weak scaling over ranks: at N ranks the job is the configuration with an N times
    # finer energy mesh; shard.plan gives each rank its wave-rotated share of the energy blocks (PAPER.md:116,
    # :135-137, Fig. 1), i.e. the configuration's own n_E per wave and rank.  No data-path collective.
    # --scaling strong splits the configuration's own energy blocks over the ranks instead (total work fixed).
    wl_job = job_workload(args, world)
    n_e_job = wl_job.n_energies()
    job_description = workload_description(args.config, wl_job)
    wl = rank_workload(wl_job, rank, world)
    hdat = args.w_layout == "channels"
    layout = rmat.PSTGF_W_CHANNEL_CONTIGUOUS if hdat else rmat.PSTGF_W_POLE_CONTIGUOUS

    def dev_W(w):
        """W on the device in the chosen memory order; an odd fastest dimension (config 6's n_poles, an odd n_chan in
        the H.DAT order) gets an even row pitch so that the TMA staging path applies."""
        Wh = np.ascontiguousarray(w.W.T) if hdat else w.W
        rows, cols = Wh.shape
        if cols % 2 == 0:
            return torch.from_numpy(Wh).cuda()
        buf = torch.zeros((rows, cols + 1), dtype=torch.float64, device="cuda")
        buf[:, :cols].copy_(torch.from_numpy(Wh))
        return buf[:, :cols]

    dev_waves, shared = [], {}
    for w in wl.waves:
        key = id(w.energies)
        if key not in shared:
            shared[key] = torch.from_numpy(w.energies).cuda()
        R = torch.empty((w.n_E, w.n_chan, w.n_chan), dtype=torch.float64, device="cuda")
        dev_waves.append((dev_W(w), torch.from_numpy(w.E_k).cuda(), shared[key], w.a, R, layout))
    single = len(dev_waves) == 1
    if not single:
        arr = rmat.make_wave_array(dev_waves)
        ws = torch.empty(rmat.pstgf_rmat_batch_workspace_bytes(arr), dtype=torch.uint8, device="cuda")
    flush_buf = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2

    sliced = args.variant == "sliced"
    if sliced:
        if not single or hdat:
            raise SystemExit("--variant sliced: single-wave configs with pole-contiguous W only")
        w0 = wl.waves[0]
        sliced_ws = torch.empty(int(rmat.load().pstgf_rmat_sliced_workspace_bytes(w0.n_chan, w0.n_poles, w0.n_E, args.slices)),
                                dtype=torch.uint8, device="cuda")

    def step():
        if sliced:
            W, E_k, en, a, R, _ = dev_waves[0]
            rmat.pstgf_rmat_form_sliced(W, E_k, en, a, n_slices=args.slices, R_out=R, workspace=sliced_ws)
            return 1 + 2 * -(-w0.n_E // max(1, min(w0.n_E, (1 << 30) // (args.slices * (-(-w0.n_chan // 128) * 128) * (-(-w0.n_poles // 64) * 64)))))
        if single:
            W, E_k, en, a, R, _ = dev_waves[0]
            (rmat.pstgf_rmat_form_hdat if hdat else rmat.pstgf_rmat_form)(W, E_k, en, a, R_out=R)
        else:
            rmat.pstgf_rmat_form_batch(arr, ws)
        return rmat.pstgf_last_launch_count()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(3, args.warmup)):
        flush_buf.zero_()
        step()
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.15)
    starts = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    ends = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    launches = 0
    barrier()
    wall0 = time.perf_counter()
    for i in range(args.steps):
        flush_buf.zero_()                 # L2 flush between timed iterations (outside the event pair)
        starts[i].record()
        launches += step()
        ends[i].record()
    barrier()
    wall = time.perf_counter() - wall0
    step_ms = [s.elapsed_time(e) for s, e in zip(starts, ends)]
    clocks = sampler.stop() if rank == 0 else None
    total_ms = float(sum(step_ms))
    t = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms_max = float(t.item())
    ms_per_step = total_ms_max / args.steps
    n_e = wl.n_energies()                       # this rank's share
    value = n_e_job * args.steps / (total_ms_max * 1e-3)
    flop = wl.counted_flop()

    # ---- dominant kernel: the persistent DMMA SYRK kernel is the only launch of a step ----
    kern_ms = total_ms / args.steps                      # this rank's average launch duration (CUDA events, launch stream)
    achieved_tflops = flop / (kern_ms * 1e-3) / 1e12
    # FP64 peak: probe the DMMA pipe (the instruction the kernel issues) right here, burst, best of 5
    probe = None
    if rank == 0:
        from paper_1909_07321_b200.measure import probe as probe_lib      # libpstgf_probe.so: bench-side, not the product
        sms = torch.cuda.get_device_properties(local_rank).multi_processor_count
        sink = torch.empty(sms * 4 * 256, dtype=torch.float64, device="cuda")
        probe = {}
        for kind, name in ((0, "dmma"), (1, "dfma"), (2, "dmma+dfma")):
            best = 0.0
            for _ in range(5):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                fl = probe_lib.fp64_probe(kind, 2000, sms * 2, 256, sink)
                e1.record()
                torch.cuda.synchronize()
                best = max(best, fl / (e0.elapsed_time(e1) * 1e-3) / 1e12)
            probe[name] = best
        # dependent-issue latency of DMMA.8x8x4 in SM clocks: one chain per warp, one warp per sub-partition
        it_chain = 2000
        best_ms = 1e30
        for _ in range(3):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            probe_lib.fp64_probe(3, it_chain, sms, 128, sink)
            e1.record()
            torch.cuda.synchronize()
            best_ms = min(best_ms, e0.elapsed_time(e1))
        dmma_latency_clk = best_ms * 1e-3 * peaks["sm_max_mhz"] * 1e6 / (it_chain * 32)
    context = None
    if rank == 0 and args.probe_i8:
        isink = torch.zeros(sms, dtype=torch.int32, device="cuda")
        best = 0.0
        for _ in range(4):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            ops = probe_lib.i8_probe(4000, sms, isink)
            e1.record()
            torch.cuda.synchronize()
            best = max(best, ops / (e0.elapsed_time(e1) * 1e-3) / 1e15)
        context = {"int8_tensor_pops": best, "kind": "tcgen05.mma.cta_group::1.kind::i8 128x256x32, operands in shared memory, "
                                                        "accumulators in TMEM, one CTA per SM (burst, best of 4)"}
    # Peak: the FP64 tensor (DMMA) rate measured live by the probe above (burst, this kernel is timed alone);
    # MEASURED_PEAKS.json has no FP64 entry.  The guide's rule (another dtype's measured peak x nominal ratio)
    # gives a LOWER figure because the bf16 measurement is power-limited (1335 MHz) while FP64 runs at 1965 MHz;
    # the harder denominator is used and the rule-based one is reported beside it.
    peak_rule = peaks["bf16"] * FP64_OVER_BF16_NOMINAL
    peak_nominal = 148 * 64 * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12      # 64 FP64 FMA/clk/SM (B300_MICROARCH.md), 37.2 TFLOP/s
    if probe and probe["dmma"] > 0:
        peak, peak_source = max(probe["dmma"], peak_rule), "DMMA.8x8x4 register-resident probe, measured in this run (burst, best of 5)"
    else:
        peak, peak_source = max(peak_nominal, peak_rule), "148 SM x 64 FMA/clk x 2 x sm_max_mhz (no probe on this rank)"
    t_fp64 = flop / (peak * 1e12)
    t_hbm = wl.r_bytes() / (peaks["hbm_gbs"] * 1e9)
    roofline = {"bound": "tensor", "achieved": achieved_tflops, "peak": peak, "unit": "TFLOP/s",
                "frac": achieved_tflops / peak, "traffic": None, "peak_source": peak_source,
                "peak_rule_bf16_x_ratio": peak_rule, "peak_nominal_fp64": peak_nominal,
                "kernel": "rmat_persistent_kernel" if not sliced else "slice_kernel + sliced_gemm_kernel (variant)", "flop_per_launch": flop,
                "t_roof_ms": 1e3 * max(t_fp64, t_hbm), "hbm_write_gbs": wl.r_bytes() / (kern_ms * 1e-3) / 1e9,
                "hbm_peak_gbs": peaks["hbm_gbs"]}
    if probe:
        roofline["fp64_probe_tflops"] = probe                       # TFLOP/s per probe kind, nothing else
        roofline["dmma_dependent_latency_clk"] = dmma_latency_clk   # a latency in SM clocks: a key of its own
    roofline["traffic"] = ncu_traffic(args.config) if not (args.n_E or sliced) else None
    roofline["traffic_source"] = ("committed ncu --set full capture (profiles/traffic.csv): DRAM bytes read + written "
                                  "per launch; not measured in this run") if roofline["traffic"] is not None else None

    # ---- end to end: HOST buffers through the C ABI, copies inside the timed region ----
    e2e = None
    if not args.no_e2e and not sliced:
        host = []
        for w in wl.waves:
            hW = torch.from_numpy(np.ascontiguousarray(w.W.T) if hdat else w.W).pin_memory()
            hEk = torch.from_numpy(w.E_k).pin_memory()
            hEn = torch.from_numpy(w.energies).pin_memory()
            hR = torch.empty((w.n_E, w.n_chan, w.n_chan), dtype=torch.float64).pin_memory()
            host.append((hW, hEk, hEn, w.a, hR, layout))
        h2d = sum(8 * (a[0].numel() + a[1].numel() + a[2].numel()) for a in host)
        d2h = sum(8 * a[4].numel() for a in host)
        e2e_steps = max(1, min(args.steps, 5 if args.config != 6 else 2))
        for _ in range(2):
            rmat.pstgf_rmat_form_batch_host(host, max_chunk_bytes=args.e2e_chunk_mib << 20)    # warm-up (allocator pool, pinned pages touched)
        barrier()
        t0 = time.perf_counter()
        e2e_launches, e2e_ms = 0, []
        for _ in range(e2e_steps):
            t1 = time.perf_counter()
            rmat.pstgf_rmat_form_batch_host(host, max_chunk_bytes=args.e2e_chunk_mib << 20)    # synchronises before returning
            e2e_ms.append(1e3 * (time.perf_counter() - t1))
            e2e_launches += rmat.pstgf_last_launch_count()
        torch.cuda.synchronize()
        dt = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(dt, op=dist.ReduceOp.MAX)
        e2e = {"value": n_e_job * e2e_steps / float(dt.item()), "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "steps": e2e_steps, "ms_per_step": 1e3 * float(dt.item()) / e2e_steps,
               "step_ms_min_max": [min(e2e_ms), max(e2e_ms)], "gpu_launches": e2e_launches,
               "api": "pstgf_rmat_form_batch_host (pinned host buffers; whole R copied back)"}
        del host

    prior = None
    if rank == 0 and world == 1 and args.prior_art:
        lib_R = [d[4][:16].cpu() for d in dev_waves]       # the library's R of the energies the comparator forms
        del dev_waves
        torch.cuda.empty_cache()
        prior = prior_art_leg(wl, library_R=lib_R)
        if not prior["max_rel_err_vs_library"] <= 1e-11:
            raise RuntimeError(f"prior-art comparator disagrees with the library: {prior['max_rel_err_vs_library']:.3e}")

    # the other BASELINE.json configurations and the few-energy shapes of config 5's wave, so that every fraction
    # DESIGN.md quotes has a twin in the driver's record (default run only: config 5, one GPU, the DMMA path)
    all_configs = None
    if rank == 0 and world == 1 and args.config == 5 and not args.n_E and not sliced and not args.no_all_configs and probe:
        try:
            del dev_waves
        except NameError:
            pass
        torch.cuda.empty_cache()
        all_configs = []
        for cfg, n_E in ((1, None), (2, None), (3, None), (4, None), (5, 1), (5, 32)):
            all_configs.append(quick_config_line(cfg, n_E, roofline["peak"], flush_buf, local_rank))
            torch.cuda.empty_cache()

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(wl, args.cpu_seconds)

    # BASELINE.md section 1 holds one published number for this metric: 14-18 s per R-matrix formation at exactly
    # config 6's shape (GPU model not stated, CUDA Fortran) -> at best 1/14 energies/s.  Context, not
    # the target; null for every other workload.
    vs_baseline = value / PAPER_ENERGIES_PER_S if (args.config == 6 and world == 1) else None
    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(3, args.warmup), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": args.scaling,
                "vs_baseline": vs_baseline, "dtype": "f64", "data": "synthetic",
                "config": job_description,           # the same dict as --impl reference prints
                "run": {"n_energies_per_rank": n_e, "l2": "flushed between timed steps (512 MiB write)",
                        "w_layout": args.w_layout, "tail_policy": args.tail_policy, "slab_policy": args.slab_policy,
                        "variant": args.variant if not sliced else f"sliced (INT8 tcgen05, {args.slices} slices): NOT the product's path",
                        "sha256": wl_job.sha256()[:16]},
                "tflops_counted": wl_job.counted_flop() * args.steps / (total_ms_max * 1e-3) / 1e12,
                "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches,
                **({"prior_art": prior} if prior else {}), **({"context": context} if context else {}),
                **({"all_configs": all_configs} if all_configs else {}),
                "clocks": clocks, "wall_s_timed_region": wall, "step_ms_min_max": [min(step_ms), max(step_ms)]}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
