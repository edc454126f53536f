#!/usr/bin/env python
"""bench.py -- headline benchmark of the limited-1PN hot path (BASELINE.json: fp64 pair-interactions/s
and RK4 steps/s at N = 1+16383, % of the B200 FP64 FMA peak).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload config2|config3|...]

One timed "step" = one classical-RK4 step of the whole path (4 force evaluations: star-star pair kernel S1 +
fused BH/1PN/RK4 epilogue S2-S4); the timed region is bracketed by the 1PN energy S5 at its start and end as in
the paper's timing runs, and those two evaluations are INSIDE the timed region.
value = ordered star-star pair interactions of the K steps / timed region (energy pairs not counted).
Prints ONE JSON line (rank 0).  Multi-GPU = independent replicas: weak scaling.
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
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

# fp64 star-star kernels by pn_get_pair_config()["variant"]: name, FP64-pipe instructions per ORDERED pair in the shipped
# SASS (cuobjdump-verified; the library reports the same number), executed flops per ordered pair (FMA = 2, MUL/ADD = 1):
#   0 tiled:     3 DADD + 9 DFMA + 3 DMUL = 15 per ordered pair (+1 MUFU.RSQ64H)
#   2 symmetric: 3 DADD + 12 DFMA + 5 DMUL = 20 per UNORDERED pair (+1 MUFU.RSQ64H) = 10 per ordered pair
#   4 symmetric, equal-mass form (every star has the same mass, as in every BASELINE.json config): the two mass
#     multiplications go: 3 DADD + 12 DFMA + 3 DMUL = 18 per unordered pair = 9 per ordered pair
#   5 ordered pairs with the Cross terms of Eq. 2.6 (--cross): 36 DADD + 124 DFMA + 56 DMUL per 4 pairs = 54 per ordered pair
#   6 the same plus the O(N^2) sum of Eq. 2.3 (--cross full): 59 per ordered pair
#   8 / 9 the Cross terms on every UNORDERED pair (pair_cross_sym_kernel, N_s >= 6144): 768 DFMA + 176 DADD + 272 DMUL per 16
#     unordered pairs = 38 per ordered pair (42 with the sum of Eq. 2.3: 832 + 192 + 320); 10 / 11: the equal-mass form of the
#     same kernel (the common G m applied at the flush): 736 + 208 + 240 = 37 per ordered pair (800 + 224 + 256 = 40)
#   7 small-system path (N_s < 3072): ONE cooperative launch per pn_step / pn_accel call, every ordered pair in the tiled
#     kernel's 15-instruction form; there is no separate pair stage to time, the launch is the whole call
PAIR_KERNELS = {0: ("pair_fp64_kernel", 15, 24.0), 2: ("pair_sym_fp64_kernel", 10, 16.0),
                4: ("pair_sym_fp64_kernel<EQM>", 9, 15.0), 5: ("pair_cross_fp64_kernel", 54, 85.0),
                6: ("pair_cross_fp64_kernel<BHX>", 59, 93.0), 7: ("small_path_kernel", 15, 24.0),
                8: ("pair_cross_sym_kernel", 38, 62.0), 9: ("pair_cross_sym_kernel<BHX>", 42, 68.0),
                10: ("pair_cross_sym_kernel<EQM>", 37, 60.0), 11: ("pair_cross_sym_kernel<BHX, EQM>", 40, 65.0),
                12: ("small_cross_kernel", 54, 85.0), 13: ("small_cross_kernel<BHX>", 59, 93.0)}
ONE_LAUNCH_PER_STEP = (7, 12, 13)  # small-system path: the launch is the whole RK4 step
SMS, FP64_LANES_PER_SM = 148, 64
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel, from the committed `ncu --set full`
# captures (per launch, cold L2: ncu flushes the caches before every replay), keyed by (variant, N_s); each entry names the
# profiles/ file (which states the command and the kernel build) it was read from.  No entry -> "traffic": null.
NCU_DRAM_BYTES_PER_PAIR_LAUNCH = {
    (4, 16383): (826624 + 185856, "profiles/r2_ncu_summary.md section 6 (r2_bench_c2, pair_sym_fp64_kernel<4,1,12,0,1,0,8,16>, round-2 build)"),
    (4, 65535): (3268864 + 142611968, "profiles/r2_ncu_summary.md section 6 (r2_bench_c3, pair_sym_fp64_kernel<4,4,3,0,1,0,8,16>, round-2 build)"),
}


def algorithmic_bytes_per_pair_launch(cfg: dict):
    """What one launch of the star-star kernel has to move by design, keyed on the kernel variant: every j record once and
    the partial sums it hands to the epilogue.  fp64 / fp32-pair hot path (variants 0 - 4): 48 B JRec per padded star, 3
    doubles per star and slot.  Cross kernels (5, 6, 8 - 11): 112 B CRec per padded star, 7 doubles per star and slot (a^SS,
    X, S), 8 with the sum U of Eq. 2.3 (variants 6, 9, 11).  Small-system path (7, 12, 13): no partial sums in global memory
    and no separate pair launch -- null."""
    v, npad, slots = cfg["variant"], cfg["padded_stars"], cfg["j_splits"]
    if v in ONE_LAUNCH_PER_STEP:
        return None
    if v in (0, 1, 2, 3, 4):
        rec, comps = 48, 3
    elif v in (5, 8, 10):
        rec, comps = 112, 7
    elif v in (6, 9, 11):
        rec, comps = 112, 8
    else:
        return None
    return {"record_bytes": rec, "sum_components": comps, "jrec_read": rec * npad, "partial_sums_written": 8 * comps * slots * npad,
            "total": rec * npad + 8 * comps * slots * npad}


_BENCH_LIB = None


def bench_lib():
    """libpn_bench.so (include/pn_bench.h): pipe-peak probes; not part of the product library."""
    global _BENCH_LIB
    if _BENCH_LIB is None:
        import ctypes

        from paper_1801_07986_b200 import build

        lib = ctypes.CDLL(str(build.BENCH_LIB))
        lib.pn_bench_fp64_peak.argtypes = [ctypes.c_void_p, ctypes.POINTER(ctypes.c_double)]
        lib.pn_bench_fp32_peak.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.POINTER(ctypes.c_double)]
        lib.pn_bench_operand_probe.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_double)]
        _BENCH_LIB = lib
    return _BENCH_LIB


def measure_fp64_peak(stream) -> float:
    import ctypes

    t = ctypes.c_double(0.0)
    rc = bench_lib().pn_bench_fp64_peak(ctypes.c_void_p(stream.cuda_stream), ctypes.byref(t))
    return t.value if rc == 0 else None


def measure_fp32_peak(stream, packed: bool) -> float:
    import ctypes

    t = ctypes.c_double(0.0)
    rc = bench_lib().pn_bench_fp32_peak(ctypes.c_void_p(stream.cuda_stream), int(packed), ctypes.byref(t))
    return t.value if rc == 0 else None


def run_probes(args) -> None:
    """--probes: the operand-bandwidth micro-probes behind DESIGN.md section 6.1 (libpn_bench.so), one JSON line each: SM cycles
    per DFMA warp-instruction and sub-partition (issue limit 2.0) for FP64 operand patterns, and for a two-register DFMA stream
    with other-pipe instructions mixed in (what a second register operand of a non-FP64 instruction costs the FP64 stream)."""
    import ctypes

    import torch

    torch.cuda.set_device(0)
    st = ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    cases = [(0, 0, 0, "DFMA, 2 distinct register operands"), (0, 1, 0, "DFMA, 3 distinct register operands"),
             (0, 2, 0, "pairs a += K d (3 reads), b -= K d (d, K from the reuse cache)"),
             (0, 3, 0, "3-register DFMA alternating with a 1-register DMUL"), (0, 4, 0, "1, 1, 3, 3 register operands"),
             (1, 0, 0, "2-register DFMA stream alone")]
    for nx in (4, 8):
        cases += [(1, 1, nx, "+ SHFL.IDX, lane in a register (2 reads)"), (1, 2, nx, "+ SHFL.BFLY, immediate mask (1 read)"),
                  (1, 3, nx, "+ IMAD (3 reads)"), (1, 4, nx, "+ MOV immediate (0 reads)"), (1, 5, nx, "+ LOP3 with immediate (1 read)"),
                  (1, 6, nx, "+ FADD (2 reads)"), (1, 7, nx, "+ LDS.128 (1 read)")]
    base = None
    for kind, mode, nx, what in cases:
        c = ctypes.c_double(0.0)
        rc = bench_lib().pn_bench_operand_probe(st, kind, mode, nx, ctypes.byref(c))
        line = {"probe": what, "kind": kind, "mode": mode, "other_per_16_dfma": nx, "cycles_per_dfma_per_subpartition": c.value if rc == 0 else None}
        if kind == 1 and nx == 0:
            base = c.value
        if kind == 1 and nx and base and rc == 0:
            line["fp64_cycles_lost_per_other_instruction"] = (c.value - base) * 16.0 / nx
        print(json.dumps(line), flush=True)


def load_peaks() -> dict:
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            return json.loads(p.read_text())
        except Exception:
            pass
    return {}


def make_problem(name: str, rank: int = 0):
    from paper_1801_07986_b200 import inputs

    if name.startswith("config"):
        p = inputs.config(int(name[6:]))
    elif name.startswith("ball"):
        p = inputs.uniform_ball_bh(int(name[4:]))
        p.dt, p.nsteps = 1e-4, 10
    else:
        raise SystemExit(f"unknown workload {name}")
    if rank:  # replicas: same recipe, different seed per rank
        seed = p.meta["seed"] + 1000 * rank
        if p.meta["model"] == "plummer+bh":
            q = inputs.plummer_bh(p.n_stars, seed, M=float(p.mass[0]), c=p.c, softening=p.softening, dt=p.dt, nsteps=p.nsteps)
        elif p.meta["model"].startswith("bahcall"):
            q = inputs.cusp_bh(p.n_stars, seed)
        else:
            q = p
        q.name = p.name
        p = q
    return p


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append((time.perf_counter(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, power, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        rows = [l for (t, l) in self.lines if t0 <= t <= t1] or [l for (_, l) in self.lines]
        for l in rows:
            f = [x.strip() for x in l.split(",")]
            try:
                sm.append(float(f[0])), smax.append(float(f[1])), power.append(float(f[2]))
            except (ValueError, IndexError):
                continue
            for nm, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


class NvmlSampler:
    """Same quantities through NVML, polled every ~2 ms from a thread: the timed region of the default run lasts
    only tens of milliseconds, too short for nvidia-smi's 100 ms loop."""

    def __init__(self, index: int):
        import pynvml

        self.nv = pynvml
        pynvml.nvmlInit()
        try:
            import torch

            uuid = str(torch.cuda.get_device_properties(index).uuid)
            self.h = pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + uuid) if not uuid.startswith("GPU-") else uuid)
        except Exception:
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
        self.samples, self.run = [], False

    def start(self):
        self.run = True
        self.thread = threading.Thread(target=self._poll, daemon=True)
        self.thread.start()

    def _poll(self):
        nv = self.nv
        while self.run:
            try:
                sm = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                try:
                    rs = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    rs = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                pw = nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0
                self.samples.append((time.perf_counter(), sm, rs, pw))
            except Exception:
                pass
            time.sleep(0.002)

    def stop(self, t0: float, t1: float) -> dict:
        nv = self.nv
        self.run = False
        self.thread.join(timeout=1.0)
        rows = [s for s in self.samples if t0 <= s[0] <= t1] or self.samples
        smax = nv.nvmlDeviceGetMaxClockInfo(self.h, nv.NVML_CLOCK_SM)
        bits = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4}
        reasons = sorted(nm for nm, b in bits.items() if any(r[2] & b for r in rows))
        return {"sm_mhz": float(np.median([r[1] for r in rows])) if rows else None, "sm_max_mhz": float(smax),
                "sm_mhz_min": float(min(r[1] for r in rows)) if rows else None,
                "power_w_max": max((r[3] for r in rows), default=None),
                "power_w_mean": float(np.mean([r[3] for r in rows])) if rows else None, "samples": len(rows), "reasons": reasons,
                "source": "nvml, 2 ms poll during the timed region"}


def make_sampler(index: int):
    try:
        return NvmlSampler(index)
    except Exception:
        return ClockSampler(index)


# ---------------------------------------------------------------------------------------------------------
# CPU oracle legs (the only places bench.py executes oracle/)
# ---------------------------------------------------------------------------------------------------------
def oracle_step_sample(p, o, rows):
    """One bounded 'step' of the oracle: a full RK4 step when all rows are taken, else 4 force evaluations
    (one RK4 step's worth) restricted to `rows`; returns pairs visited."""
    if rows is None:
        o.step(p.pos, p.vel, p.dt, 1)
        return 4 * p.pairs_per_eval
    for _ in range(4):
        o.accel_rows(p.pos, p.vel, rows)
    return 4 * len(rows) * (p.n_stars - 1)


def oracle_rows(p, budget_pairs=3.0e9):
    """All stars if one RK4 step stays under the pair budget (config 2 does), else a seeded subset of i-rows."""
    if 4 * p.pairs_per_eval <= budget_pairs:
        return None, "full RK4 steps (all rows)"
    r = max(64, int(budget_pairs / 4 / (p.n_stars - 1)))
    rows = np.sort(np.random.default_rng(12345).choice(np.arange(1, p.N), size=r, replace=False))
    return rows, f"4 force evaluations per step on a seeded subset of {r} of {p.n_stars} i-rows, each against all j"


def cpu_baseline(p, target_s=12.0, max_steps=200, terms=0) -> dict:
    from oracle.pn_oracle import Oracle

    o = Oracle(p.mass, p.G, p.c, p.softening, kind="fast", terms=terms)
    rows, what = oracle_rows(p)
    pairs, t0, n = 0, time.perf_counter(), 0
    while n < max_steps and (time.perf_counter() - t0 < target_s or n == 0):
        pairs += oracle_step_sample(p, o, rows)
        n += 1
    dt = time.perf_counter() - t0
    out = {"value": pairs / dt, "unit": "pair-interactions/s", "cores": o.max_threads, "kind": "oracle",
           "build": "oracle/pn_oracle.c -DORACLE_FAST (double, -O3 -march=native, OpenMP over i)",
           "note": "the parity oracle as it stands: plain scalar loops over every ORDERED pair, array-of-structures data, a sqrt and "
                   "three divisions per pair, no use of Newton's third law -- a reported baseline, not a tuned CPU code; a ratio "
                   "against it says nothing about kernel quality (the roofline fraction does)",
           "sample": f"{n} x {what}; {dt:.1f} s", "steps_per_s": (n / dt) if rows is None else None}
    # the like-for-like counterpart of the paper's single-core CPU column (Table 3.2): the same oracle on
    # ONE thread, on a seeded subset of i-rows (rows are independent), about 5 s
    n_all = o.max_threads
    o1 = Oracle(p.mass, p.G, p.c, p.softening, kind="fast", terms=terms, threads=1)
    rows1, _ = oracle_rows(p, budget_pairs=6.0e8 / (8.0 if terms else 1.0))
    if rows1 is None:
        rows1 = np.arange(1, p.N)
    t0 = time.perf_counter()
    pairs1 = oracle_step_sample(p, o1, rows1)
    dt1 = time.perf_counter() - t0
    o1.lib.oracle_set_threads(n_all)
    out["one_core"] = {"value": pairs1 / dt1, "unit": "pair-interactions/s", "cores": 1,
                       "sample": f"4 force evaluations on a seeded subset of {len(rows1)} of {p.n_stars} i-rows; {dt1:.1f} s"}
    return out


def run_reference(args) -> None:
    """--impl reference: the oracle, as it stands, on the host cores; same metric/config keys as our arm."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle.pn_oracle import Oracle

    p = make_problem(args.workload)
    o = Oracle(p.mass, p.G, p.c, p.softening, kind="fast", terms=cross_mask(args))
    # bound the whole run to ~4e10 pair visits (about 1.5 min on 8 cores) whatever K is
    rows, what = oracle_rows(p, budget_pairs=max(2.0e8, 4.0e10 / max(1, args.steps)))
    for _ in range(args.warmup):
        oracle_step_sample(p, o, rows if rows is None else rows[:64])
    pairs, t0 = 0, time.perf_counter()
    for _ in range(args.steps):
        pairs += oracle_step_sample(p, o, rows)
    dt = time.perf_counter() - t0
    val = pairs / dt
    line = {
        "impl": "reference", "metric": "fp64 pair-interactions/s", "value": val, "unit": "pair-interactions/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(p, args),
        "cpu_baseline": {"value": val, "unit": "pair-interactions/s", "cores": o.max_threads, "kind": "oracle",
                         "sample": f"each step = {what}"},
        "e2e": {"value": val, "unit": "pair-interactions/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def max_over_ranks(values, world: int, device):
    """Per-rank timings -> the slowest rank's (the contract's max over ranks); any torch.distributed backend."""
    import torch

    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist

        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def whole_job_rate(world: int, steps: int, pairs_per_step: int, seconds: float) -> float:
    """Replicas only: every rank processes the same number of pairs; the job's rate is all of them
    over the slowest rank's time."""
    return world * steps * pairs_per_step / seconds


def cross_mask(args) -> int:
    """PN_OPT_CROSS_TERMS value (== the oracle's terms mask): 0, 1 = Eq. 2.6, 3 = Eqs. 2.6 + 2.3."""
    return {None: 0, "star": 1, "full": 3}[getattr(args, "cross", None)]


def workload_config(p, args) -> dict:
    return {"workload": p.name, "N": p.N, "n_stars": p.n_stars, "pairs_per_force_eval": p.pairs_per_eval,
            "force_evals_per_step": 4, "dt": p.dt, "c": p.c, "softening": p.softening, "M": float(p.mass[0]),
            "integrator": "classical RK4", "energy_evals_in_timed_region": 2,
            "force": {None: "hot path (north_star)", "star": "hot path + [a_i]_Cross (Eq. 2.6)",
                      "full": "hot path + [a_i]_Cross (Eq. 2.6) + [a_1]_Cross (Eq. 2.3): the paper's full limited-1PN force"}[
                          getattr(args, "cross", None)],
            "l2": "flushed (256 MiB write) between timed steps, outside the per-step event pairs",
            "parallelism": f"replicas x{args.gpus}" if args.gpus > 1 else "single GPU"}


# ---------------------------------------------------------------------------------------------------------
# Our arm: the CUDA path through the C-ABI
# ---------------------------------------------------------------------------------------------------------
def run_ours(args) -> None:
    import torch
    import torch.distributed as dist

    from paper_1801_07986_b200 import PN, binding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    p = make_problem(args.workload, rank)
    K, W = args.steps, max(3, args.warmup)
    stream = torch.cuda.current_stream()
    pn = PN(p.mass, p.G, p.c, p.softening, stream=stream)
    if args.cross:
        pn.pn_set_option(binding.PN_OPT_CROSS_TERMS, cross_mask(args))
    cfg = pn.pn_get_pair_config()
    pos_d, vel_d = torch.from_numpy(p.pos).cuda(), torch.from_numpy(p.vel).cuda()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")  # > 126 MB L2

    # ---------------- device-resident timing: energy, K x (RK4 step), energy; per-item CUDA event pairs
    # pn_step stays on its CUDA graph; event-record nodes bracket the pair stage of the first force evaluation of every
    # step (every 4th launch of the dominant kernel: bracketing all four costs 5 % of the step in event overhead)
    pn.pn_set_option(binding.PN_OPT_TIME_PAIR, 2)
    pn.pn_set_state(pos_d, vel_d)
    for _ in range(W):
        pn.pn_step(p.dt, 1)
    pn.pn_energy()
    pn.pn_set_state(pos_d, vel_d)
    pn.pn_get_pair_time(reset=True)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K + 2)]
    sampler = make_sampler(local)
    sampler.start()
    time.sleep(0.25)
    barrier()
    launches0 = pn.pn_get_launch_count()
    t_wall0 = time.perf_counter()
    ev[0][0].record(stream)
    e_start = pn.pn_energy()
    ev[0][1].record(stream)
    for k in range(K):
        flush.zero_()
        ev[k + 1][0].record(stream)
        pn.pn_step(p.dt, 1)
        ev[k + 1][1].record(stream)
    flush.zero_()
    ev[K + 1][0].record(stream)
    e_end = pn.pn_energy()
    ev[K + 1][1].record(stream)
    barrier()
    t_wall1 = time.perf_counter()
    launches = pn.pn_get_launch_count() - launches0
    clocks = sampler.stop(t_wall0, t_wall1)
    ms_items = [a.elapsed_time(b) for a, b in ev]
    ms_energy = ms_items[0] + ms_items[-1]
    ms_steps = sum(ms_items[1:-1])
    ms_total = ms_energy + ms_steps
    pair_ms, pair_n = pn.pn_get_pair_time(reset=True)
    pn.pn_set_option(binding.PN_OPT_TIME_PAIR, 0)
    dfma_peak = measure_fp64_peak(stream)  # register-only DFMA chains on this device, TFLOP/s (libpn_bench.so)

    # ---------------- same K steps through the CUDA-graph path (information: what a user gets by default)
    pn.pn_set_state(pos_d, vel_d)
    pn.pn_step(p.dt, 16 + 1)
    barrier()
    g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    g0.record(stream)
    pn.pn_step(p.dt, K)
    g1.record(stream)
    barrier()
    ms_graph = g0.elapsed_time(g1)

    # ---------------- end to end through the host-buffer entry points: every step copies its inputs H2D from
    # pinned memory and reads its result (the new state) back D2H
    hp, hv = torch.from_numpy(p.pos).pin_memory(), torch.from_numpy(p.vel).pin_memory()
    ho_p, ho_v = torch.empty_like(hp).pin_memory(), torch.empty_like(hv).pin_memory()
    for _ in range(2):
        pn.pn_set_state_host(hp, hv)
        pn.pn_step(p.dt, 1)
        pn.pn_get_state_host(ho_p, ho_v)
    barrier()
    t0 = time.perf_counter()
    for _ in range(K):
        pn.pn_set_state_host(hp, hv)
        pn.pn_step(p.dt, 1)
        pn.pn_get_state_host(ho_p, ho_v)
    barrier()
    e2e_s = time.perf_counter() - t0

    # ---------------- max over ranks, whole-job aggregate
    pairs_per_step = 4 * p.pairs_per_eval
    ms_total_m, ms_steps_m, e2e_m, ms_graph_m, ms_energy_m = max_over_ranks([ms_total, ms_steps, e2e_s, ms_graph, ms_energy], world, "cuda")
    # `value` must not depend on --steps: the timed region holds K steps and 2 energy evaluations, the workload as stated
    # (BASELINE.json: p.nsteps steps, E at the start and at the end) holds 2 per p.nsteps steps.  One step is therefore charged
    # its own measured time plus 2 / p.nsteps of a measured energy evaluation, whatever K was; the raw sums are reported too.
    ms_step_charged = ms_steps_m / K + (ms_energy_m / 2) * (2.0 / p.nsteps)
    value = whole_job_rate(world, 1, pairs_per_step, ms_step_charged * 1e-3)
    e2e_val = whole_job_rate(world, K, pairs_per_step, e2e_m)

    if rank == 0:
        peaks = load_peaks()
        sm_max = peaks.get("sm_max_mhz", 1965.0)
        peak_tflops = SMS * FP64_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
        pair_avg_ms = pair_ms / max(1, pair_n)
        kname, instr, exec_flops = PAIR_KERNELS[cfg["variant"]]
        assert instr == cfg["fp64_instr_per_pair"]
        pairs_per_launch = p.pairs_per_eval
        if cfg["variant"] in ONE_LAUNCH_PER_STEP:  # one launch = one whole RK4 step (4 force evaluations): its time is the step's
            pair_avg_ms, pair_n, pairs_per_launch = ms_steps / K, K, 4 * p.pairs_per_eval
        kernel_pairs_per_s = pairs_per_launch / (pair_avg_ms * 1e-3) if pair_n else None
        achieved = kernel_pairs_per_s * 2 * instr / 1e12 if pair_n else None
        roof = {
            "bound": "alu", "kernel": kname, "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
            "frac": (achieved / peak_tflops) if achieved else None,
            "traffic": NCU_DRAM_BYTES_PER_PAIR_LAUNCH.get((cfg["variant"], p.n_stars), (None, None))[0],
            "traffic_source": NCU_DRAM_BYTES_PER_PAIR_LAUNCH.get((cfg["variant"], p.n_stars), (None, "no ncu capture of this kernel at this size"))[1],
            "algorithmic_bytes": algorithmic_bytes_per_pair_launch(cfg),
            "convention": f"{instr} FP64-pipe instructions per ordered pair in the shipped SASS, each counted as an "
                          f"FMA (2 flops) = FP64-pipe issue-slot utilisation; peak = {SMS} SMs x {FP64_LANES_PER_SM} FP64 lanes x 2 x "
                          f"{sm_max:.0f} MHz (clocks.max.sm; no measured fp64 peak in MEASURED_PEAKS.json)",
            "pairs_per_launch": pairs_per_launch, "avg_launch_ms": pair_avg_ms, "launches_timed": pair_n,
            "launches_in_timed_steps": K if cfg["variant"] in ONE_LAUNCH_PER_STEP else 4 * K,
            "pair_kernel_share_of_steps": (1.0 if cfg["variant"] in ONE_LAUNCH_PER_STEP else 4 * K * pair_avg_ms / ms_steps) if ms_steps else None,
            "kernel_pairs_per_s": kernel_pairs_per_s,
            "frac_at_sampled_clock": (achieved / (peak_tflops * clocks["sm_mhz"] / sm_max)) if achieved and clocks.get("sm_mhz") else None,
            "executed_flops_frac": (kernel_pairs_per_s * exec_flops / 1e12 / peak_tflops) if achieved else None,
            "classic_20flop_frac": (kernel_pairs_per_s * 20.0 / 1e12 / peak_tflops) if achieved else None,
            "peak_measured_dfma": dfma_peak,
            "frac_of_measured_dfma": (achieved / dfma_peak) if achieved and dfma_peak else None,
        }
        bar = bar_leg(args, stream, flush, local, peak_tflops, sm_max, dfma_peak) if (world == 1 and args.workload == "config2" and not args.cross and not args.no_bar) else None
        sustained = ([sustained_leg(w, stream, local, peak_tflops, args.sustain_s) for w in ("config2", "config3")]
                     if (world == 1 and args.workload == "config2" and not args.cross and not args.no_bar and args.sustain_s > 0) else None)
        small = small_leg(stream) if (world == 1 and args.workload == "config2" and not args.cross and not args.no_bar) else None
        base = cpu_baseline(p, terms=cross_mask(args)) if not args.no_cpu_baseline else None
        line = {
            "metric": "fp64 pair-interactions/s", "value": value, "unit": "pair-interactions/s", "n_gpus": world,
            "steps": K, "warmup": W, "ms_per_step": ms_step_charged, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": workload_config(p, args),
            "steps_per_s": world / (ms_step_charged * 1e-3), "rk4_only_ms_per_step": ms_steps_m / K,
            "energy_ms_per_eval": ms_energy_m / 2, "timed_region_ms": ms_total_m,
            "value_definition": f"pairs of one RK4 step / (measured ms per step + 2/{p.nsteps} of a measured pn_energy): the workload as "
                                f"stated has 2 energy evaluations per {p.nsteps} steps; independent of --steps",
            "graph_ms_per_step": ms_graph_m / K,
            "graph_pairs_per_s": whole_job_rate(world, K, pairs_per_step, ms_graph_m * 1e-3),
            "energy_drift": (e_end - e_start) / abs(e_start), "pair_config": cfg,
            "clocks": clocks,
            "e2e": {"value": e2e_val, "unit": "pair-interactions/s", "h2d_bytes_per_step": 2 * p.N * 24,
                    "d2h_bytes_per_step": 2 * p.N * 24, "ms_per_step": 1e3 * e2e_m / K,
                    "api": "pn_set_state_host + pn_step + pn_get_state_host per step, pinned host buffers"},
            "gpu_launches": launches, "roofline": roof, "bar": bar, "sustained": sustained, "config1": small, "cpu_baseline": base,
        }
        print(json.dumps(line), flush=True)
    pn.pn_destroy()
    if world > 1:
        dist.destroy_process_group()


def small_leg(stream, steps: int = 200) -> dict:
    """BASELINE.json configs[0] (N = 1+1023), the small-system path: one pn_step(dt, steps) call = one cooperative launch."""
    import torch

    from paper_1801_07986_b200 import PN

    p = make_problem("config1")
    pn = PN(p.mass, p.G, p.c, p.softening, stream=stream)
    cfg = pn.pn_get_pair_config()
    pn.pn_set_state(torch.from_numpy(p.pos).cuda(), torch.from_numpy(p.vel).cuda())
    pn.pn_step(p.dt, 8)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(stream)
    pn.pn_step(p.dt, steps)
    b.record(stream)
    torch.cuda.synchronize()
    ms = a.elapsed_time(b) / steps
    launches = pn.pn_get_launch_count()
    pn.pn_destroy()
    return {"workload": p.name, "N": p.N, "pair_config": cfg, "steps": steps, "ms_per_step": ms, "steps_per_s": 1e3 / ms,
            "pairs_per_s": 4 * p.pairs_per_eval / (ms * 1e-3), "launches_for_all_steps": launches - 2,
            "note": "one cooperative launch runs all steps (small_path_kernel); round 1: 0.0462 ms per step with 8 launches per step"}


def sustained_leg(workload: str, stream, local, peak_tflops, seconds: float) -> dict:
    """>= `seconds` of back-to-back pn_step on the batched CUDA graph (what a production run does; PAPER.md:130 times
    32-step runs, PAPER.md:172 runs 1.3 M steps), clocks / power / throttle reasons sampled over the whole leg, then -- with no
    pause -- a short instrumented stretch (event-record nodes around the pair stage of the first force evaluation of every
    step) for the pair kernel's in-graph fraction of the FP64 issue roofline under the same thermal state."""
    import torch

    from paper_1801_07986_b200 import PN, binding

    p = make_problem(workload)
    pn = PN(p.mass, p.G, p.c, p.softening, stream=stream)
    cfg = pn.pn_get_pair_config()
    kname, instr, exec_flops = PAIR_KERNELS[cfg["variant"]]
    pn.pn_set_state(torch.from_numpy(p.pos).cuda(), torch.from_numpy(p.vel).cuda())
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(stream)
    pn.pn_step(p.dt, 32)
    b.record(stream)
    torch.cuda.synchronize()
    est = a.elapsed_time(b) / 32
    steps = int(math.ceil(seconds * 1e3 / est / 16.0)) * 16
    sampler = make_sampler(local)
    sampler.start()
    t0 = time.perf_counter()
    a.record(stream)
    pn.pn_step(p.dt, steps)
    b.record(stream)
    torch.cuda.synchronize()  # the option drops the captured graphs: not while they run (the rebuild idles the GPU for a few ms)
    pn.pn_set_option(binding.PN_OPT_TIME_PAIR, 2)
    n_inst = max(8, min(200, steps // 10))
    pn.pn_step(p.dt, n_inst)
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    clocks = sampler.stop(t0, t1)
    ms = a.elapsed_time(b) / steps
    pair_ms, pair_n = pn.pn_get_pair_time(reset=True)
    pn.pn_destroy()
    avg = pair_ms / max(1, pair_n)
    rate = p.pairs_per_eval / (avg * 1e-3) if pair_n else None
    return {"workload": p.name, "N": p.N, "kernel": kname, "steps": steps, "seconds": a.elapsed_time(b) * 1e-3, "ms_per_step": ms,
            "steps_per_s": 1e3 / ms, "pairs_per_s": 4 * p.pairs_per_eval / (ms * 1e-3),
            "step_frac": 4 * p.pairs_per_eval / (ms * 1e-3) * 2 * instr / 1e12 / peak_tflops,
            "pair_stage": {"launches_timed": pair_n, "avg_launch_ms": avg, "kernel_pairs_per_s": rate,
                           "frac": (rate * 2 * instr / 1e12 / peak_tflops) if rate else None,
                           "executed_flops_frac": (rate * exec_flops / 1e12 / peak_tflops) if rate else None,
                           "note": f"{n_inst} instrumented steps right after the sustained stretch (a few ms of graph rebuild in between)"},
            "clocks": clocks,
            "note": "batched CUDA graph (16 steps per launch), no L2 flush, no energy evaluation; step_frac = whole step against the "
                    "pair kernel's issue roofline (epilogues and launch gaps count as loss)"}


def bar_leg(args, stream, flush, local, peak_tflops, sm_max, dfma_peak=None, steps: int = 3) -> dict:
    """The configuration the >= 70 % bar of north_star is defined on (BASELINE.json configs[2], N = 1+65535): a short leg of
    the same measurement (RK4 steps on the CUDA graph, the pair stage of the first force evaluation of every step bracketed
    by event-record nodes, L2 flushed between steps, clocks sampled), so that the driver's own run observes it."""
    import torch

    from paper_1801_07986_b200 import PN, binding

    p = make_problem("config3")
    pn = PN(p.mass, p.G, p.c, p.softening, stream=stream)
    cfg = pn.pn_get_pair_config()
    kname, instr, exec_flops = PAIR_KERNELS[cfg["variant"]]
    pn.pn_set_option(binding.PN_OPT_TIME_PAIR, 2)
    pn.pn_set_state(torch.from_numpy(p.pos).cuda(), torch.from_numpy(p.vel).cuda())
    pn.pn_step(p.dt, 3)
    torch.cuda.synchronize()
    pn.pn_get_pair_time(reset=True)
    sampler = make_sampler(local)
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    t0 = time.perf_counter()
    for a, b in ev:
        flush.zero_()
        a.record(stream)
        pn.pn_step(p.dt, 1)
        b.record(stream)
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    clocks = sampler.stop(t0, t1)
    ms_steps = [a.elapsed_time(b) for a, b in ev]
    pair_ms, pair_n = pn.pn_get_pair_time(reset=True)
    pn.pn_destroy()
    avg = pair_ms / max(1, pair_n)
    rate = p.pairs_per_eval / (avg * 1e-3)
    return {"workload": p.name, "N": p.N, "kernel": kname, "pair_config": cfg, "steps": steps, "ms_per_step": float(np.mean(ms_steps)),
            "pairs_per_s": 4 * p.pairs_per_eval / (float(np.mean(ms_steps)) * 1e-3), "avg_launch_ms": avg, "launches_timed": pair_n,
            "kernel_pairs_per_s": rate, "frac": rate * 2 * instr / 1e12 / peak_tflops, "peak": peak_tflops, "unit": "TFLOP/s",
            "executed_flops_frac": rate * exec_flops / 1e12 / peak_tflops, "classic_20flop_frac": rate * 20.0 / 1e12 / peak_tflops,
            "peak_measured_dfma": dfma_peak, "frac_of_measured_dfma": (rate * 2 * instr / 1e12 / dfma_peak) if dfma_peak else None,
            "convention": f"frac: {instr} FP64-pipe instructions per ordered pair, issue-slot convention (every DADD / DMUL counted as an FMA), "
                          f"as roofline.frac -- the convention the >= 70 % bar is claimed in (north_star: 'FP64 FMA-pipe utilisation'); "
                          f"executed_flops_frac counts {exec_flops:.0f} executed flops per ordered pair (FMA = 2, MUL / ADD = 1)", "clocks": clocks}


def run_sweep(args) -> None:
    """--sweep: BASELINE.json config 5 (and configs 2-4 when --sweep-configs): ONE force evaluation per size and per
    pair precision, pairs/s and % of the FMA roofline versus N.  One JSON line per case (not the default bench line)."""
    import torch

    from paper_1801_07986_b200 import PN, binding, inputs

    torch.cuda.set_device(0)
    stream = torch.cuda.current_stream()
    peaks = load_peaks()
    sm_max = peaks.get("sm_max_mhz", 1965.0)
    peak64 = SMS * FP64_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    peak32 = SMS * 128 * 2 * sm_max * 1e6 / 1e12
    cases = [("ball%d" % k, lambda k=k: inputs.uniform_ball_bh(k)) for k in range(args.kmin, args.kmax + 1)]
    if args.sweep_configs:
        cases += [("config%d" % i, lambda i=i: inputs.config(i)) for i in (1, 2, 3, 4)]
    for name, make in cases:
        p = make()
        pn = PN(p.mass, p.G, p.c, p.softening, stream=stream)
        pos, vel = torch.from_numpy(p.pos).cuda(), torch.from_numpy(p.vel).cuda()
        acc = torch.empty_like(pos)
        pn.pn_set_option(binding.PN_OPT_TIME_PAIR, 1)
        # third leg: the first NEXT row of the scope table, [a_i]_Cross (Eq. 2.6) fused into an fp64 ordered-pair kernel
        for prec, pname, peak, cross in ((binding.PN_FP64, "fp64", peak64, 0), (binding.PN_FP32_PAIR, "fp32pair", peak32, 0),
                                         (binding.PN_FP64, "fp64+cross", peak64, binding.PN_CROSS_STAR),
                                         (binding.PN_FP64, "fp64+cross_full", peak64, binding.PN_CROSS_STAR | binding.PN_CROSS_BH)):
            pn.pn_set_option(binding.PN_OPT_PAIR_PRECISION, prec)
            pn.pn_set_option(binding.PN_OPT_CROSS_TERMS, cross)
            instr = pn.pn_get_pair_config()["fp64_instr_per_pair"]  # pipe instructions per ordered pair of the kernel in use
            reps = 5 if p.n_stars < 200000 else 2
            for _ in range(2):
                pn.pn_accel(pos, vel, acc)
            pn.pn_get_pair_time(reset=True)
            ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
            for a, b in ev:
                a.record(stream)
                pn.pn_accel(pos, vel, acc)
                b.record(stream)
            torch.cuda.synchronize()
            ms = float(np.median([a.elapsed_time(b) for a, b in ev]))
            pair_ms, n = pn.pn_get_pair_time(reset=True)
            pair_ms = pair_ms / n if n else ms  # small-system path: no separate pair stage, the evaluation is one launch
            tfl = p.pairs_per_eval * 2 * instr / (pair_ms * 1e-3) / 1e12
            epi = None
            cfg = pn.pn_get_pair_config()
            if cross == 0 and prec == binding.PN_FP64 and cfg["variant"] not in ONE_LAUNCH_PER_STEP:
                # the O(N) kernel of the hot path (fused S2 + S3 + S4 epilogue) inside captured RK4 steps: the interval between two
                # bracketed pair stages.  Design bytes: the partial sums it reduces (24 B per star and slot) + the per-star state
                # it reads and writes (stages 0 - 2: 216, 264, 264 B); algorithmic bytes: SURVEY.md 8(d), ~100 B per body.
                dt = getattr(p, "dt", None) or 1e-4
                pn.pn_set_state(pos, vel)
                pn.pn_step(dt, 1)
                pn.pn_get_pair_time(reset=True), pn.pn_get_epilogue_time(reset=True)
                pn.pn_step(dt, 3)
                e_ms, e_n = pn.pn_get_epilogue_time(reset=True)
                pn.pn_get_pair_time(reset=True)
                if e_n:
                    t = e_ms / e_n * 1e-3
                    design = 24 * cfg["j_splits"] * cfg["padded_stars"] + 248 * p.n_stars
                    hbm = peaks.get("hbm_gbs", 6549.4)
                    epi = {"kernel": "epilogue_kernel<MODE_RK4>", "intervals": e_n, "avg_ms": e_ms / e_n, "design_bytes": design,
                           "algorithmic_bytes": 100 * p.N, "gbs_design": design / t / 1e9, "gbs_algorithmic": 100 * p.N / t / 1e9,
                           "hbm_peak_gbs": hbm, "frac_of_hbm_design": design / t / 1e9 / hbm,
                           "note": "interval between two bracketed pair stages of a captured RK4 step (one epilogue launch + its launch "
                                   "gaps); L2-resident below N ~ 2^18, HBM-bound only at the largest sizes"}
            print(json.dumps({
                "workload": name, "N": p.N, "precision": pname, "pairs": p.pairs_per_eval, "accel_ms": ms,
                "accel_pairs_per_s": p.pairs_per_eval / (ms * 1e-3), "pair_kernel_ms": pair_ms,
                "pair_kernel_pairs_per_s": p.pairs_per_eval / (pair_ms * 1e-3), "pipe_instr_per_pair": instr,
                "roofline_frac": tfl / peak, "peak_tflops": peak, "epilogue": epi, "pair_config": cfg}), flush=True)
        pn.pn_destroy()


def run_variants(args) -> None:
    """--variants: the table behind choose_sym's size thresholds (pn_api.cu): every form of the symmetric fp64 pair kernel
    (PN_SYM_FORM = w1: one-warp blocks on 128-star tiles, js: four warps share one 128 x 128 tile pair, u512: 512-star tiles),
    forced through the environment of pn_create, at sizes around the switch points; pair-stage time of one force evaluation,
    median of 7.  One JSON line per (N, form); "auto" is what the library picks by itself."""
    import torch

    from paper_1801_07986_b200 import PN, binding, inputs

    torch.cuda.set_device(0)
    stream = torch.cuda.current_stream()
    sm_max = load_peaks().get("sm_max_mhz", 1965.0)
    peak64 = SMS * FP64_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    for n_stars in (4095, 8191, 12287, 15359, 16383, 20479, 32767, 36863, 49151, 65535, 131071):
        p = inputs.plummer_bh(n_stars, seed=n_stars)
        pos, vel = torch.from_numpy(p.pos).cuda(), torch.from_numpy(p.vel).cuda()
        acc = torch.empty_like(pos)
        for form in ("auto", "w1", "js", "u512"):
            os.environ.pop("PN_SYM_FORM", None)
            if form != "auto":
                os.environ["PN_SYM_FORM"] = form
            pn = PN(p.mass, p.G, p.c, p.softening, stream=stream)
            os.environ.pop("PN_SYM_FORM", None)
            pn.pn_set_option(binding.PN_OPT_PAIR_KERNEL, binding.PN_PAIR_SYMMETRIC)
            pn.pn_set_option(binding.PN_OPT_TIME_PAIR, 1)
            cfg = pn.pn_get_pair_config()
            times = []
            for r in range(9):
                pn.pn_accel(pos, vel, acc)
                ms, n = pn.pn_get_pair_time(reset=True)
                if r >= 2:
                    times.append(ms / n)
            pn.pn_destroy()
            ms = float(np.median(times))
            print(json.dumps({"N": p.N, "form": form, "pair_kernel_ms": ms, "pair_kernel_pairs_per_s": p.pairs_per_eval / (ms * 1e-3),
                              "roofline_frac": p.pairs_per_eval * 2 * cfg["fp64_instr_per_pair"] / (ms * 1e-3) / 1e12 / peak64,
                              "pair_config": cfg}), flush=True)


# PAPER.md:137-142, Table 3.2: elapsed seconds of 32 RK4 steps + energy at both ends, mean of 10 samples,
# N: (CPU+GPU [Tesla K20c via Goose], CPU only [one core of an i7-3770K])
PAPER_TABLE_3_2 = {100: (1.5392, 0.3479), 300: (1.9651, 3.0501), 1000: (1.941, 33.652), 3000: (5.0517, 302.31),
                   10000: (38.934, 3358.6), 30000: (339.956, 30188.0)}


def run_paper_timing(args) -> None:
    """The paper's timing experiment with its full limited-1PN force (Eqs. 2.1-2.6) through the C-ABI: per N, 10 samples of
    [pn_energy, pn_step(dt, 32), pn_energy], device-resident state, wall clock around the three calls (pn_energy
    synchronises).  Context against another machine's numbers, not a target."""
    import torch

    from paper_1801_07986_b200 import PN, binding, inputs

    torch.cuda.set_device(0)
    for n_total, (t_gpu_paper, t_cpu_paper) in PAPER_TABLE_3_2.items():
        p = inputs.cold_shell_bh(n_total, seed=n_total)
        pn = PN(p.mass, p.G, p.c, p.softening, stream=torch.cuda.current_stream())
        pn.pn_set_option(binding.PN_OPT_CROSS_TERMS, binding.PN_CROSS_STAR | binding.PN_CROSS_BH)
        pos, vel = torch.from_numpy(p.pos).cuda(), torch.from_numpy(p.vel).cuda()
        samples, drift = [], None
        for rep in range(12):  # 2 warm-up + 10 samples
            pn.pn_set_state(pos, vel)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            e0 = pn.pn_energy()
            pn.pn_step(p.dt, 32)
            e1 = pn.pn_energy()
            dt = time.perf_counter() - t0
            if rep >= 2:
                samples.append(dt)
            drift = (e1 - e0) / abs(e0)
        mean, sd = float(np.mean(samples)), float(np.std(samples, ddof=1))
        print(json.dumps({
            "workload": "paper_timing (PAPER.md:130-144, Table 3.2)", "N": n_total, "rk4_steps": 32, "energy_evals": 2,
            "force": "full limited 1PN (Eqs. 2.1-2.6)", "elapsed_s_mean": mean, "elapsed_s_sd": sd, "samples": len(samples),
            "energy_drift_32_steps": drift, "paper_elapsed_s_k20c": t_gpu_paper, "paper_elapsed_s_cpu_1core": t_cpu_paper,
            "paper_hardware": "Tesla K20c + Core i7-3770K (Goose 1.3.3)", "ratio_vs_paper_gpu": t_gpu_paper / mean,
            "ratio_vs_paper_cpu": t_cpu_paper / mean, "pair_config": pn.pn_get_pair_config(),
            "note": "initial conditions of the paper's timing runs are not given; cold shell of PAPER.md:152-160"}), flush=True)
        pn.pn_destroy()


def run_cold_collapse(args) -> None:
    """The paper's test model (Fig. 2): N = 10^4 bodies, cold shell 1 < r < 10, M = 100 m = 0.01,
    c = G = 1, softening 1e-3, classical RK4 with dt = 2^k, full limited-1PN force; relative energy error against t.
    The paper reports about 1e-2 at t = 10, nearly independent of dt in {2^-17, 2^-16, 2^-15} (its
    figures are missing from the extraction).  One JSON line per output time."""
    import torch

    from paper_1801_07986_b200 import PN, binding, inputs

    torch.cuda.set_device(0)
    p = inputs.cold_shell_bh(args.collapse_n, seed=0)
    dt = 2.0 ** args.dt_log2
    pn = PN(p.mass, p.G, p.c, p.softening, stream=torch.cuda.current_stream())
    if not args.collapse_hot_path:
        pn.pn_set_option(binding.PN_OPT_CROSS_TERMS, binding.PN_CROSS_STAR | binding.PN_CROSS_BH)
    pn.pn_set_state(torch.from_numpy(p.pos).cuda(), torch.from_numpy(p.vel).cuda())
    e0 = pn.pn_energy()
    chunk = max(1, int(round(args.collapse_every / dt)))
    n_chunks = int(round(args.t_end / (chunk * dt)))
    t_wall = time.perf_counter()
    for k in range(1, n_chunks + 1):
        pn.pn_step(dt, chunk)
        e = pn.pn_energy()
        x, v = pn.pn_get_state()
        r = torch.linalg.norm(x[1:] - x[0], dim=1)
        print(json.dumps({"workload": "cold_collapse (PAPER.md:152-176)", "N": p.N, "dt_log2": args.dt_log2,
                          "force": "hot path" if args.collapse_hot_path else "full limited 1PN (Eqs. 2.1-2.6)",
                          "t": k * chunk * dt, "steps": k * chunk, "energy": e, "rel_energy_error": (e - e0) / abs(e0),
                          "r_min_to_bh": float(r.min()), "r_median": float(r.median()),
                          "wall_s": time.perf_counter() - t_wall}), flush=True)
    pn.pn_destroy()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--variants", action="store_true", help="forms of the symmetric fp64 pair kernel around choose_sym's thresholds")
    ap.add_argument("--sweep", action="store_true", help="config-5 single-evaluation sweep (one JSON line per case)")
    ap.add_argument("--sweep-configs", action="store_true")
    ap.add_argument("--kmin", type=int, default=10)
    ap.add_argument("--kmax", type=int, default=20)
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50, help="timed RK4 steps (default: the 50 steps BASELINE.json configs[1] states)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config2")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sustain-s", type=float, default=2.0, help="length of each sustained leg (config 2 and config 3) in seconds; 0: skip")
    ap.add_argument("--no-bar", action="store_true", help="skip the short config-3 leg (the >= 70 %% bar's configuration)")
    ap.add_argument("--cross", nargs="?", const="star", default=None, choices=["star", "full"],
                    help="add the Cross terms (NEXT rows of the scope table): star = [a_i]_Cross, Eq. 2.6; "
                         "full = also [a_1]_Cross, Eq. 2.3 (the paper's full limited-1PN force)")
    ap.add_argument("--cold-collapse", action="store_true", help="the paper's test model: energy error against t (JSON lines)")
    ap.add_argument("--collapse-n", type=int, default=10000)
    ap.add_argument("--dt-log2", type=int, default=-15)
    ap.add_argument("--t-end", type=float, default=10.0)
    ap.add_argument("--collapse-every", type=float, default=0.25, help="output interval in time units")
    ap.add_argument("--collapse-hot-path", action="store_true", help="without the Cross terms")
    ap.add_argument("--probes", action="store_true", help="operand-bandwidth micro-probes of DESIGN.md section 6.1 (JSON lines)")
    ap.add_argument("--paper-timing", action="store_true",
                    help="the paper's timing experiment (PAPER.md:130-144, Table 3.2): 32 RK4 steps + 2 energy evaluations of "
                         "the full limited-1PN force at N = 100 ... 30000, one JSON line per N")
    args = ap.parse_args()
    if args.probes:
        run_probes(args)
    elif args.cold_collapse:
        run_cold_collapse(args)
    elif args.paper_timing:
        run_paper_timing(args)
    elif args.variants:
        run_variants(args)
    elif args.sweep:
        run_sweep(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
