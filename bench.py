#!/usr/bin/env python
"""bench.py -- throughput of the tetrahedron-DOS hot path (arxiv 1710.10789) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg4] [--impl ours|reference]

A "step" is one pass of the whole hot path (implicit cube/tetrahedron indexing,
corner sort, energy window, corner weights Eq. 11-15, orbital projection, accumulation, fp64 merge +
prefix sum) over one synthetic workload -- by default BASELINE.json configs[3] (the headline roofline
config: seeded 8-orbital model, Nk=128, 4000 energies), inputs already resident in HBM.

Prints ONE JSON line (rank 0).  `value` = nominal (tetrahedron, band, omega) evaluations per second,
n_tb*nE / t, the paper's accounting (every energy of every (tetrahedron, band));
`effective_evals_per_s` counts only the n_eval evaluations with E1 < omega < E4 the method needs.
`roofline` is the main kernel against the FP32-ALU peak; `e2e` is the same
metric through the C-ABI call with HOST buffers (H2D + kernels + D2H inside the timed region);
`cpu_baseline` is the fp64 oracle on this box's host cores on a bounded sample of the same workload.

--impl reference times the oracle (the only "reference" this paper-only tier has) on the same config,
each step a bounded sample.  N > 1 (torchrun): the cubes are sharded in z-slabs, one rank per GPU,
each rank's additive fp64 partial is all-reduced (NCCL) and finalised -- strong scaling.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1710_10789_b200 import workloads as wl  # noqa: E402  (input generators only)

# Algorithmic flop models.
# Paper formulation (Eq. 12-14 weights per energy, then the orbital loop): per in-window evaluation
# F_eval = 40 + 18*norb (weights case-averaged + 2*4*norb FMAs + 2*norb adds), per (tetrahedron, band)
# F_tb = 40 + 5*norb (sort, differences, reciprocals, Eq.-15 sum).
def flops_alg(n_eval: int, n_tb: int, norb: int) -> float:
    return float(n_eval) * (40 + 18 * norb) + float(n_tb) * (40 + 5 * norb)


# Formulation of main kernel generation 5 (recounted, as SURVEY.md 8(d) requires when the formulation changes:
# algorithmic flops may not exceed executed flops).  Low/high evaluations (Eq. 12/14 with H, J hoisted):
# T and D each 2 FMAs per orbital + 8 flops for the powers of s -> 8*norb + 8.  Mid evaluations (Eq. 13):
# ~70 flops for the eight weights + 2*(2*4*norb) for the projection (the accumulation rides on the FMAs).
# Per (tetrahedron, band): 40 + 5*norb as above + H, J of the two outer intervals, 2 * 11*norb.
def flops_alg_gen5(n_eval: int, n_mid: int, n_tb: int, norb: int) -> float:
    return (float(n_eval - n_mid) * (8 * norb + 8) + float(n_mid) * (70 + 16 * norb)
            + float(n_tb) * (40 + 5 * norb + 22 * norb))


# FP32-ALU peak derived from the guide's unit counts and clocks: SMs x 128 FP32 lanes x 2 flops (FMA)
# x max SM clock (B200_PROFILING.md: 148 SMs, clocks.max.sm 1965 MHz).
def fp32_peak_tflops(num_sms: int, sm_max_mhz: float) -> float:
    return num_sms * 128 * 2 * sm_max_mhz * 1e6 / 1e12


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="cfg4", choices=sorted(wl.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--layout", default="aos", choices=["aos", "soa"],
                    help="aos: E[ik][n], W[ik][n][m] (default); soa: E[n][ik], W[n][m][ik] (k fastest; 1 GPU only)")
    ap.add_argument("--op", default="dos", choices=["dos", "eigh", "h2dos", "weights", "select", "table2"],
                    help="dos: the hot path (the contract's JSON line).  The others time the SURVEY 8(f) operations on "
                         "one GPU and print their own JSON line(s): eigh (tetra_eigh), h2dos (H(k) -> eigh -> DOS on the "
                         "device), weights (tetra_weights), select (5 orbitals + total), table2 (the paper's Table II "
                         "shapes: device-resident, host buffers, one-shot)")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--oracle-single-core", action="store_true",
                    help="with --impl reference: one thread on 1/8 of the sample (the cpu_baseline leg's single-core figure)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-fp64", action="store_true", help="skip the fp64-accumulation variant's cost")
    ap.add_argument("--cache", default=os.environ.get("TDOS_CACHE", "/tmp/tdos_cache"))
    return ap.parse_args()


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.01):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        self.period = period_s
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake_slowdown",
        }
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(self.period)

    def start(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self) -> dict:
        self._stop.set()
        if self._thr is not None:
            self._thr.join()
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


# ----------------------------------------------------------------------------------------------
# The oracle legs (the ONLY places bench.py touches oracle/): cpu_baseline and --impl reference.
# ----------------------------------------------------------------------------------------------
def oracle_sample_planes(cfg) -> int:
    """Bounded sample of the workload: the cubes of the first N3/16 z-planes (>= 1)."""
    return max(1, cfg.nk[2] // 16)


def run_oracle_sample(cfg, E, W, om, reps: int = 1, warmup: int = 0, single_core: bool = False):
    """Time the fp64 oracle, as it stands, on the sample.  Returns (median seconds per rep, n_tb, n_eval, cores, text).
    single_core: one thread on 1/8 of the sample's planes (comparable in spirit with the paper's single-core
    CPU reference)."""
    import oracle
    oracle.build()
    planes = oracle_sample_planes(cfg)
    if single_core:
        planes = max(1, planes // 8)
    hi = cfg.nk[0] * cfg.nk[1] * planes
    cores = 1 if single_core else min(oracle.max_threads(), len(os.sched_getaffinity(0)))
    Wn = None if cfg.model == "cosine" else W
    times, res = [], None
    for r in range(warmup + reps):
        t0 = time.perf_counter()
        res = oracle.tetra_dos(E, Wn, cfg.nk, om, windowed=True, nthreads=cores, cube_range=(0, hi))
        if r >= warmup:
            times.append(time.perf_counter() - t0)
    text = ("oracle.tetra_dos(windowed=True: Eq. 12-14 inside (E1,E4), Eq. 15 by step+prefix), fp64, OpenMP over cubes, "
            "on the cubes of z-planes [0,%d) of %s (%d of %d cubes), all %d energies"
            % (planes, cfg.name, hi, int(np.prod(cfg.nk)), cfg.nE))
    return float(np.median(times)), res["n_tb"], res["n_eval"], cores, text


def cpu_model() -> str:
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.startswith("model name"):
                return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def reference_arm(args, cfg, rank: int):
    """--impl reference: the oracle on host cores, rank 0 only."""
    if rank != 0:
        return
    E, W, om = wl.make_inputs(cfg, args.cache)
    sec, n_tb, n_eval, cores, text = run_oracle_sample(cfg, E, W, om, reps=args.steps, warmup=args.warmup,
                                                       single_core=args.oracle_single_core)
    value = n_tb * cfg.nE / sec
    line = {
        "impl": "reference", "metric": "tetra*band*omega evaluations/sec", "value": value, "unit": "eval/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec * 1e3,
        "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(cfg, args.gpus, args.layout),
        "effective_evals_per_s": n_eval / sec, "seconds": sec,
        "cpu_baseline": {"value": value, "unit": "eval/s", "cores": cores, "kind": "oracle", "sample": text,
                         "timing": "median of %d after %d warm-up" % (args.steps, args.warmup), "cpu": cpu_model()},
        "e2e": {"value": value, "unit": "eval/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def hbm_peak_gbs():
    """(GB/s, source): the measured copy bandwidth of this pool's B200s, else the profiling guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs"
    except Exception:
        return 6650.0, "of fallback (B200_PROFILING.md: 6.65 TB/s)"


def run_ops(args, cfg):
    """--op eigh | h2dos | weights | select | table2: the SURVEY.md 8(f) operations on one GPU, timed with CUDA events
    after 3 warm-ups, inputs resident on the device unless the line says otherwise; one JSON line per operation."""
    import torch
    from paper_1710_10789_b200 import binding
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    peak, peak_src = hbm_peak_gbs()
    K, Wm = args.steps, max(args.warmup, 3)

    def timed(fn, steps=K):
        for _ in range(Wm):
            fn()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(steps):
            fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / steps

    def out(line):
        line.update({"n_gpus": 1, "steps": K, "warmup": Wm, "data": "synthetic"})
        print(json.dumps(line), flush=True)

    nk, nb, norb, nE = cfg.nk, cfg.nb, cfg.norb, cfg.nE
    nkt = int(np.prod(nk))
    if args.op in ("eigh", "h2dos"):
        assert cfg.model == "tb8", "--op eigh / h2dos need an 8-orbital config"
        H = wl.tb8_hamiltonian(nk)
        dH = torch.from_numpy(H).to(dev)
        dE = torch.empty((nkt, nb), device=dev)
        dA = torch.empty((nkt, nb, nb), dtype=torch.complex64, device=dev)
        dOm = torch.from_numpy(wl.omega_grid(cfg.omega_min, cfg.omega_max, nE)).to(dev)
        dos, nos = torch.empty((norb, nE), device=dev), torch.empty((norb, nE), device=dev)
        with binding.Plan(nk, nb, norb, nE) as plan:
            ms_eigh = timed(lambda: plan.tetra_eigh(dH, dE, dA))
            bytes_alg = nkt * (nb * nb * 8 + nb * 4 + nb * nb * 8)
            roof = {"bound": "hbm", "kernel": "tdos_eigh8", "achieved": bytes_alg / ms_eigh / 1e6, "peak": peak, "unit": "GB/s",
                    "frac": bytes_alg / ms_eigh / 1e6 / peak, "traffic": None, "peak_source": peak_src,
                    "bytes_alg": bytes_alg,
                    "note": "algorithmic bytes = H in + E, A out; the kernel is fp64-ALU work (cyclic Jacobi, 8 lanes per "
                            "matrix), so the HBM fraction is a lower-bound reference, not a target"}
            if args.op == "eigh":
                out({"op": "eigh", "metric": "8x8 Hermitian eigenproblems/sec", "value": nkt / (ms_eigh * 1e-3), "unit": "matrices/s",
                     "ms_per_step": ms_eigh, "higher_is_better": True, "dtype": "f64", "config": workload_config(cfg, 1),
                     "roofline": roof, "gpu_launches": K})
                return
            ms_dos = timed(lambda: plan.tetra_dos_complex(dE, torch.view_as_real(dA), dOm, dos, nos))

            def chain():
                plan.tetra_eigh(dH, dE, dA)
                plan.tetra_dos_complex(dE, torch.view_as_real(dA), dOm, dos, nos)
            ms_chain = timed(chain)
            out({"op": "h2dos", "metric": "H(k) -> DOS grids/sec (device resident)", "value": 1e3 / ms_chain, "unit": "grids/s",
                 "ms_per_step": ms_chain, "higher_is_better": True, "dtype": "f64 eigensolver, f32 DOS",
                 "config": workload_config(cfg, 1), "eigh_ms": ms_eigh, "tetra_dos_complex_ms": ms_dos,
                 "h_bytes": int(H.nbytes), "gpu_launches": K * 6,
                 "note": "PAPER.md:289 best case: the Hamiltonian is on the device and nothing returns to the host but DOS, N"})
        return
    E, W, om = wl.make_inputs(cfg, args.cache)
    dE, dOm = torch.from_numpy(E).to(dev), torch.from_numpy(om).to(dev)
    dW = None if cfg.model == "cosine" else torch.from_numpy(W).to(dev)
    if args.op == "weights":
        nW = 16
        en = torch.from_numpy(wl.omega_grid(cfg.omega_min, cfg.omega_max, nW)).to(dev)
        wk = torch.empty((nW, nb, nkt), device=dev)
        dwk = torch.empty((nW, nb, nkt), device=dev)
        with binding.Plan(nk, nb, norb, nE) as plan:
            ms = timed(lambda: plan.tetra_weights(dE, en, wk, dwk))
        bytes_alg = E.nbytes + 2 * wk.numel() * 4           # E read once, wk and dwk written once
        out({"op": "weights", "metric": "per-k integration weights/sec", "value": 2 * wk.numel() / (ms * 1e-3), "unit": "weights/s",
             "ms_per_step": ms, "higher_is_better": True, "dtype": "f32", "config": dict(workload_config(cfg, 1), nW=nW),
             "roofline": {"bound": "hbm", "kernel": "tdos_kweights", "achieved": bytes_alg / ms / 1e6, "peak": peak, "unit": "GB/s",
                          "frac": bytes_alg / ms / 1e6 / peak, "traffic": None, "peak_source": peak_src, "bytes_alg": bytes_alg,
                          "note": "24 scalar red.global.add per output element plus the two memsets; untuned"},
             "gpu_launches": K})
        return
    if args.op == "select":
        sel = [0, 2, 3, 5, 7][:max(1, min(5, norb - 1))]
        dos, nos = torch.empty((len(sel) + 1, nE), device=dev), torch.empty((len(sel) + 1, nE), device=dev)
        dosf, nosf = torch.empty((norb, nE), device=dev), torch.empty((norb, nE), device=dev)
        with binding.Plan(nk, nb, norb, nE) as plan:
            ms_sel = timed(lambda: plan.tetra_dos_select(dE, dW, dOm, sel, True, dos, nos))
            ms_full = timed(lambda: plan.tetra_dos(dE, dW, dOm, dosf, nosf))
        out({"op": "select", "metric": "DOS grids/sec, %d orbitals + total" % len(sel), "value": 1e3 / ms_sel, "unit": "grids/s",
             "ms_per_step": ms_sel, "higher_is_better": True, "dtype": "f32", "config": workload_config(cfg, 1),
             "all_orbitals_ms": ms_full, "gpu_launches": K * 5})
        return
    # ---- table2: PAPER.md Table II (:315-320) shapes, 8 bands, 1024 energies, 5 orbitals + total
    rows = []
    for shape in ((10, 10, 10), (20, 20, 10), (25, 25, 25), (60, 60, 10)):
        n = int(np.prod(shape))
        E, W = wl.tb8_bands(shape)
        om = wl.omega_grid(-6.0, 4.0, 1024)
        dE, dW, dOm = (torch.from_numpy(a).to(dev) for a in (E, W, om))
        hE, hW, hOm = (torch.from_numpy(a).pin_memory() for a in (E, W, om))
        sel = [0, 2, 3, 5, 7]
        dos, nos = torch.empty((6, 1024), device=dev), torch.empty((6, 1024), device=dev)
        hdos, hnos = torch.empty((6, 1024)).pin_memory(), torch.empty((6, 1024)).pin_memory()
        odos, onos = np.empty((8, 1024), np.float32), np.empty((8, 1024), np.float32)
        with binding.Plan(shape, 8, 8, 1024) as plan:
            ms_dev = timed(lambda: plan.tetra_dos_select(dE, dW, dOm, sel, True, dos, nos), steps=max(K, 20))
            t = []
            for r in range(Wm + 5):
                t0 = time.perf_counter()
                plan.tetra_dos_select(hE, hW, hOm, sel, True, hdos, hnos, memspace=binding.TDOS_HOST)
                t.append((time.perf_counter() - t0) * 1e3)
            ms_host = float(np.median(t[Wm:]))
        ms_shot = None
        if shape[0] == shape[1] == shape[2]:   # tetra_dos_simple takes cubic grids only
            t = []
            for r in range(Wm + 5):   # one-shot: plan creation + H2D + kernels + D2H + destroy, pageable host arrays
                t0 = time.perf_counter()
                binding.tetra_dos_simple(E, W, shape[0], 8, 8, -6.0, 4.0, 1024, odos, onos)
                t.append((time.perf_counter() - t0) * 1e3)
            ms_shot = float(np.median(t[Wm:]))
        rows.append({"n_k": n, "grid": list(shape), "evaluations_paper": n * 6 * 8 * 1024,
                     "device_resident_ms": ms_dev, "host_buffers_ms": ms_host, "one_shot_simple_ms": ms_shot,
                     "paper_gtx970_ms": {1000: [24.4, 98.7], 4000: [81.8, 169.4], 15625: [318.9, 451.4], 36000: [732.0, 936.7]}[n]})
    out({"op": "table2", "metric": "run time per DOS grid, Table II shapes", "unit": "ms", "higher_is_better": False,
         "dtype": "f32", "rows": rows,
         "note": "5 orbitals + total, 8 bands, 1024 energies on the seeded 8-orbital model (the paper's FeSe parameters are not "
                 "available). device_resident = the paper's best case (:289), host_buffers = tetra_dos_select with pinned host "
                 "arrays on an existing plan, one_shot_simple = tetra_dos_simple (cubic grids only; all 8 orbitals; plan "
                 "creation, H2D from pageable memory, kernels, D2H, destroy: the paper's worst case, :287). "
                 "paper_gtx970_ms = [best, worst] of Table II, another machine: context only"})


def workload_config(cfg, n_gpus: int, layout: str = "aos") -> dict:
    return {"workload": "%s: %s, Nk=%dx%dx%d, nb=%d, norb=%d, nE=%d on [%g,%g]" % (
                cfg.name, "seeded 8-orbital tetragonal tight-binding" if cfg.model == "tb8" else "simple-cubic cosine band",
                cfg.nk[0], cfg.nk[1], cfg.nk[2], cfg.nb, cfg.norb, cfg.nE, cfg.omega_min, cfg.omega_max),
            "nk": list(cfg.nk), "nb": cfg.nb, "norb": cfg.norb, "nE": cfg.nE,
            "layout": "AoS E[ik][n], W[ik][n][m]" if layout == "aos" else "SoA E[n][ik], W[n][m][ik]",
            "parallelism": "1 GPU" if n_gpus == 1 else "z-slabs over %d GPUs + all-reduce of fp64 partials" % n_gpus}


# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the main kernel, from the committed
# `ncu --set full` capture (profiles/, named there); None until a capture of that config exists.
# The number is a constant from that file, NOT measured in this run: `roofline.traffic_source` names the file.
NCU_TRAFFIC_BYTES = {("cfg4", 3): (1.394956e9 + 280.968e6, "profiles/r01_v3_regions_cfg4.md"),
                     ("cfg4", 5): (739.806e6 + 81.059e6, "profiles/r03_cfg4.md"),
                     ("cfg5", 3): (2.604243e9 + 120.008e6, "profiles/r02_v3_main_cfg5.md")}


def main():
    args = parse_args()
    cfg = wl.CONFIGS[args.config]
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        reference_arm(args, cfg, rank)
        return 0
    if args.op != "dos":
        if rank == 0:
            run_ops(args, cfg)
        return 0

    import torch
    import torch.distributed as dist
    from paper_1710_10789_b200 import binding, multigpu, sharding   # raises if libtetrados.so is missing: no CPU fallback

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()

    # ---- inputs (seeded, synthetic; rank 0 diagonalises and caches, the others load the cache)
    if rank == 0:
        E, W, om = wl.make_inputs(cfg, args.cache)
    barrier()
    if rank != 0:
        E, W, om = wl.make_inputs(cfg, args.cache)
    N1, N2, N3 = cfg.nk
    nb, norb, nE = cfg.nb, cfg.norb, cfg.nE
    unitW = cfg.model == "cosine"
    z_lo, z_hi = sharding.z_slab(rank, world, N3)
    slab_local = world > 1 and z_hi > z_lo
    if slab_local:
        # a rank holds its slab's k-planes plus the halo plane and nothing else (AoS: whole planes are
        # contiguous; the halo of the last rank is plane 0)
        plane = N1 * N2
        lo, hi, h = z_lo * plane, z_hi * plane, (z_hi % N3) * plane
        E = np.concatenate([E[lo:hi], E[h:h + plane]])
        if not unitW:
            W = np.concatenate([W[lo:hi], W[h:h + plane]])
    dE = torch.from_numpy(E).to(dev)
    dW = None if unitW else torch.from_numpy(W).to(dev)
    layout = binding.TDOS_AOS
    if args.layout == "soa":   # the same numbers with k fastest (north_star (1)); converted on the device
        if world > 1:
            raise SystemExit("--layout soa is a 1-GPU measurement (the z-slab staging of the N > 1 leg slices AoS arrays)")
        layout = binding.TDOS_SOA
        dE = dE.t().contiguous()
        if dW is not None:
            dW = dW.permute(1, 2, 0).contiguous()
    dOm = torch.from_numpy(om).to(dev)
    dos = torch.zeros((norb, nE), device=dev)
    nos = torch.zeros((norb, nE), device=dev)
    part = torch.zeros((3, norb, nE), dtype=torch.float64, device=dev)
    plan = binding.Plan(cfg.nk, nb, norb, nE, device=local_rank)

    def step():
        if world == 1:
            plan.tetra_dos(dE, dW, dOm, dos, nos, layout=layout)
        else:   # partial over this rank's z-slab -> ONE all-reduce (the path's only exchange step) -> finalize
            multigpu.sharded_step(plan, dE, dW, dOm, N3, rank, world, part, dos, nos, dist.all_reduce, slab_local=slab_local)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    ev0.record()
    for _ in range(args.steps):
        step()
    ev1.record()
    torch.cuda.synchronize()
    barrier()
    clocks = sampler.stop()
    ms = torch.tensor([ev0.elapsed_time(ev1) / args.steps], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    ms_per_step = float(ms.item())

    # ---- work counters (exact integers from the kernel) and per-kernel device times of the timed steps
    main_ms, merge_ms = plan.kernel_ms(min(args.steps, 64))
    cnt = plan.last_counters()
    gen = int(cnt["kernel"])
    c = torch.tensor([cnt["n_tb"], cnt["n_eval"], max(cnt["n_eval_mid"], 0)], dtype=torch.int64, device=dev)
    if world > 1:
        dist.all_reduce(c)
        km = torch.tensor([main_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(km, op=dist.ReduceOp.MAX)
        main_ms = float(km.item())
    n_tb, n_eval, n_mid = int(c[0].item()), int(c[1].item()), int(c[2].item())
    info = plan.info()
    # kernels of this library launched per step, counted by the library itself (adaptive plans: window sample + both
    # main kernels, one of which returns at once; then merge and finalize; memsets and NCCL not counted)
    launches_per_step = int(info["launches"])

    # ---- e2e: the same step through the C-ABI with HOST (pinned) buffers
    e2e = None
    if not args.no_e2e:
        hE = (torch.from_numpy(E) if layout == binding.TDOS_AOS else dE.cpu()).pin_memory()
        hW = None if unitW else (torch.from_numpy(W) if layout == binding.TDOS_AOS else dW.cpu()).pin_memory()
        hOm = torch.from_numpy(om).pin_memory()
        hdos = torch.zeros((norb, nE)).pin_memory()
        hnos = torch.zeros((norb, nE)).pin_memory()
        plane = N1 * N2

        def e2e_step():
            if world == 1:
                plan.tetra_dos(hE, hW, hOm, hdos, hnos, layout=layout, memspace=binding.TDOS_HOST)
                return
            # each rank stages its own z-slab plus the halo plane (all its arrays hold), then partial -> all-reduce
            # -> finalize
            dE.copy_(hE, non_blocking=True)
            if hW is not None:
                dW.copy_(hW, non_blocking=True)
            dOm.copy_(hOm, non_blocking=True)
            step()
            if rank == 0:
                hdos.copy_(dos, non_blocking=True)
                hnos.copy_(nos, non_blocking=True)
            torch.cuda.synchronize()

        for _ in range(2):
            e2e_step()
        torch.cuda.synchronize()
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            e2e_step()
        torch.cuda.synchronize()
        barrier()
        t = torch.tensor([(time.perf_counter() - t0) / args.e2e_steps], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
        h2d = E.nbytes + (0 if unitW else W.nbytes) + om.nbytes      # world > 1: this rank's slab + halo plane
        if world > 1:   # whole job: every rank's arrays (the halo planes are copied twice across the job)
            tt = torch.tensor([h2d], dtype=torch.float64, device=dev)
            dist.all_reduce(tt)
            h2d = int(tt.item())
        # reference for the achieved host->device rate: ONE plain
        # cudaMemcpyAsync of the same E + W bytes from the same pinned buffers, nothing overlapped with it
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        plain = []
        for _ in range(3):
            torch.cuda.synchronize()
            c0.record()
            dE.copy_(hE, non_blocking=True)
            if hW is not None:
                dW.copy_(hW, non_blocking=True)
            c1.record()
            torch.cuda.synchronize()
            plain.append(c0.elapsed_time(c1) * 1e-3)
        copy_bytes = E.nbytes + (0 if unitW else W.nbytes)
        e2e = {"value": n_tb * nE / e2e_s, "unit": "eval/s", "ms_per_step": e2e_s * 1e3,
               "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(2 * norb * nE * 4),
               "h2d_gbs": h2d / e2e_s / 1e9,
               "h2d_gbs_plain": copy_bytes / min(plain) / 1e9, "plain_copy_ms": min(plain) * 1e3,
               "note": "h2d_gbs = staged bytes / whole e2e step (copies overlapped with the kernels); h2d_gbs_plain = one "
                       "plain cudaMemcpyAsync of the same E + W bytes from the same pinned buffers, timed alone"}

    # ---- cost of the fp64-accumulation variant on the same workload
    fp64_acc = None
    if world == 1 and not args.no_fp64:
        plan.set_accumulation(True)
        for _ in range(2):
            step()
        torch.cuda.synchronize()
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        f0.record()
        for _ in range(3):
            step()
        f1.record()
        torch.cuda.synchronize()
        fp64_acc = {"ms_per_step": f0.elapsed_time(f1) / 3, "main_kernel_ms": plan.kernel_ms(3)[0],
                    "what": "tdos_plan_set_accumulation(TDOS_ACC_FP64): single-precision corner weights, every sum after "
                            "them in fp64 (generation 3 kernel, fp64 block partials)"}
        plan.set_accumulation(True, weights_fp64=True)
        for _ in range(2):
            step()
        torch.cuda.synchronize()
        f0.record()
        for _ in range(2):
            step()
        f1.record()
        torch.cuda.synchronize()
        fp64_acc["all_fp64_ms_per_step"] = f0.elapsed_time(f1) / 2
        fp64_acc["all_fp64_what"] = "TDOS_ACC_FP64_ALL: corner weights in double precision too (agrees with the fp64 oracle to 1e-14)"
        plan.set_accumulation(False)

    # ---- roofline of the dominant kernel (tdos_main): FP32 ALU
    props = torch.cuda.get_device_properties(dev)
    sm_max = clocks.get("sm_max_mhz") or 1965.0
    peak = fp32_peak_tflops(props.multi_processor_count, sm_max)
    # `achieved` / `frac`: SURVEY.md 8(d)'s per-unit counts (the method as the paper states it) x the units the kernel
    # itself counted -- the count the north star's 60 % target is read against.  The kernel's own
    # formulation needs fewer flops (H, J hoisted for Eq. 12/14); that recount is reported beside it.
    fl_paper = flops_alg(n_eval, n_tb, norb) / world    # per launch (each rank's share on average)
    fl_kernel = flops_alg_gen5(n_eval, n_mid, n_tb, norb) / world if gen == 5 else fl_paper
    fl = fl_paper
    achieved = fl / (main_ms * 1e-3) / 1e12
    bytes_alg = 4.0 * N1 * N2 * N3 * nb * (1 + (0 if unitW else norb)) + 8.0 * norb * nE
    traffic = NCU_TRAFFIC_BYTES.get((cfg.name, gen)) if layout == binding.TDOS_AOS else None
    roofline = {"bound": "alu", "kernel": "tdos_main5" if gen == 5 else "tdos_main", "achieved": achieved, "peak": peak,
                "unit": "TFLOP/s", "frac": achieved / peak, "traffic": traffic[0] if traffic else None,
                "traffic_source": (traffic[1] + " (constant from that ncu capture, not measured in this run)") if traffic else None,
                "flop_model": "SURVEY.md 8(d): F_eval = 40 + 18 norb, F_tb = 40 + 5 norb, units counted by the kernel",
                "note": "achieved/frac count the ALGORITHMIC flops of the paper's formulation (the figure the 0.60 target is "
                        "stated in), not instructions executed: the kernel's own formulation needs fewer flops, and the "
                        "fraction of the FP32 peak it actually keeps busy is frac_kernel_formulation",
                "frac_kernel_formulation": fl_kernel / (main_ms * 1e-3) / 1e12 / peak,
                "flops_kernel_formulation_per_launch": fl_kernel,
                "frac_paper_formulation": fl_paper / (main_ms * 1e-3) / 1e12 / peak,
                "flops_paper_formulation_per_launch": fl_paper,
                "peak_source": "derived: %d SMs x 128 FP32 lanes x 2 x %.0f MHz (B200_PROFILING.md unit counts and clocks)"
                               % (props.multi_processor_count, sm_max),
                "flops_alg_per_launch": fl, "main_kernel_ms": main_ms, "merge_finalize_ms": merge_ms,
                "bytes_alg": bytes_alg, "hbm_gbs_at_main_kernel": bytes_alg / world / (main_ms * 1e-3) / 1e9}
    try:
        roofline["fma_probe_tflops"] = {"ffma": plan.fp32_fma_probe(False), "ffma2": plan.fp32_fma_probe(True)}
    except Exception as ex:   # diagnostics only
        roofline["fma_probe_tflops"] = str(ex)

    line = {
        "metric": "tetra*band*omega evaluations/sec", "value": n_tb * nE / (ms_per_step * 1e-3), "unit": "eval/s",
        "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step,
        "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": dict(workload_config(cfg, world, args.layout), l2="inputs (%.0f MB) larger than L2 (126 MB), no flush" % (bytes_alg / 1e6)
                       if bytes_alg > 126e6 else "inputs fit in L2; L2 not flushed between steps",
                       tile=list(info["tile"]), grid=info["grid"], threads=info["threads"], smem=info["smem"]),
        "effective_evals_per_s": n_eval / (ms_per_step * 1e-3), "dos_grids_per_s": 1e3 / ms_per_step,
        "n_tb": n_tb, "n_eval": n_eval, "n_eval_mid": n_mid if gen >= 4 else None, "kernel_generation": gen,
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches_per_step * args.steps, "roofline": roofline,
        "fp64_accumulation": fp64_acc,
    }

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        # The oracle is timed in a process of its own (this file's --impl reference arm: 3 warm-ups, median of 5;
        # PAPER.md:285 takes the mean of five runs for its CPU reference).  Inside this process, next to the CUDA context
        # and torch's thread pools, the same call ran a third slower than in a clean one (4.3e10 against 6.6e10 eval/s
        # on the same box), and the first ~4 calls of any process run 1.5x slower (OpenMP team start-up, first touch of
        # the thread-private histograms).  The GPU is idle meanwhile.
        import subprocess

        def oracle_leg(extra):
            cmd = [sys.executable, os.path.abspath(__file__), "--impl", "reference", "--config", cfg.name, "--steps", "5",
                   "--warmup", "3", "--cache", args.cache] + extra
            env = dict(os.environ)
            for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
                env.pop(k, None)
            r = subprocess.run(cmd, capture_output=True, text=True, env=env, timeout=900)
            if r.returncode != 0:
                raise RuntimeError("oracle leg failed: " + r.stderr[-500:])
            return json.loads(r.stdout.strip().splitlines()[-1])

        ol = oracle_leg([])
        line["cpu_baseline"] = dict(ol["cpu_baseline"], seconds=ol["seconds"], effective_evals_per_s=ol["effective_evals_per_s"],
                                    process="separate process (python bench.py --impl reference --steps 5 --warmup 3)")
        o1 = oracle_leg(["--oracle-single-core"])
        line["cpu_baseline"]["single_core"] = {"value": o1["value"], "unit": "eval/s", "cores": 1,
                                               "sample": o1["cpu_baseline"]["sample"], "seconds": o1["seconds"],
                                               "effective_evals_per_s": o1["effective_evals_per_s"]}
    if rank == 0:
        print(json.dumps(line), flush=True)
    plan.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
