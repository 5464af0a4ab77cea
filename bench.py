#!/usr/bin/env python
"""bench.py - replica-site updates/s of the PCPD multispin hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg4] [--impl ours|reference]

One STEP = one pass of the hot path over one batch of synthetic input:
`pcpd_run(SWEEPS_PER_STEP)` (RNG + masks + schedule + bitwise rule, SURVEY.md
8(a) a1-a3) followed by `pcpd_density` (a4).  Init (a5) runs once before the
warm-up and is timed separately (config.init_ms).  Workload at N = 1:
BASELINE.json configs[3] ("cfg4": L = 2^22, 2048 replicas, 1 GiB lattice,
d = 0.8, p = 0.12, full start, seed 4), the configuration the metric is quoted
on.  N > 1: every rank runs its own cfg4-sized shard of word columns
(word_offset = rank * W; no data-path collective) - weak scaling.

Prints ONE JSON line (rank 0).  See DESIGN.md section 7 for every field.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

import workloads as wl

SWEEPS_PER_STEP = 10
# dram__bytes_read.sum + dram__bytes_write.sum of one sweep launch, a CONSTANT copied from the committed
# `ncu --set full` capture named beside it (not measured by this run; re-captured when the kernel changes)
NCU_TRAFFIC_BYTES = {"cfg4": (2.088e9, "profiles/r2_sweep_kernel_full.md: 1.074 GB read + 1.014 GB written per launch")}
METRIC = "replica_site_updates_per_sec"
UNIT = "replica-site updates/s"


# --------------------------------------------------------------------------
# Algorithmic instruction count per attempt-word (SURVEY.md
# 8(d)): fixed part F + per-Philox-block cost * lazily-needed blocks, where the
# number of blocks needed to decide all 64 lanes of a generic mask is
# sum_m [1 - (1 - 4^-m)^64] (a lane stays undecided after k planes w.p. 2^-k).
def blocks_needed_generic(nplanes: int) -> float:
    nblk_max = (nplanes + 1) // 2
    return sum(1.0 - (1.0 - 4.0 ** (-m)) ** 64 for m in range(nblk_max))


def nplanes_of(q: float) -> int:
    T = int(math.floor(math.ldexp(q, 32)))
    if T == 0 or T >= 1 << 32:
        return 0
    return 32 - ((T & -T).bit_length() - 1)


# Per-block and fixed thread-instruction counts of the sweep kernel's own SASS (sweep_warp_device.cuh, nvcc 12.9):
# one strength-reduced Philox-4x32-10 block = 16 IMAD.WIDE.U32 + 18 LOP3; MSB-first compare of its two planes with T
# = 8 instructions (per plane and 32-lane half one LOP3 for the und chain + one 32-bit IMAD for the signed-sum lt;
# the run-time specialised kernel needs 4 in its prefix - the yardstick keeps the generic 8).  The MISC block has no
# threshold compare (Fm = ~lo folds into the rule's truth tables); the ANNI block of the paper's annihilation mask
# takes 4 LOP3 (two planes ANDed and gated, per half) instead of a compare.  Per attempt: 2 IMAD.WIDE (slot
# constants) + 1 IMAD.HI (position) and ~40 logic/address ops (rule 22, position/seam/address 12, tail masks 6; TCPD +6).
WIDE_PER_BLOCK, LOP_PER_BLOCK, CMP_PER_BLOCK, PMASK_PER_BLOCK = 16.0, 18.0, 8.0, 4.0
WIDE_FIXED = 3.0


def algorithmic_instr_per_attempt_word(cfg: wl.Config) -> dict:
    alu_fixed = 40.0 if (cfg.variant & 0xff) == wl.PCPD else 46.0
    npd, npp = nplanes_of(cfg.d), nplanes_of(cfg.p)
    raw = WIDE_PER_BLOCK + LOP_PER_BLOCK        # a block whose planes are used as they are (MISC)
    cmp_blk = raw + CMP_PER_BLOCK               # a block whose two planes are compared with T
    fixed = WIDE_FIXED + alu_fixed
    if cfg.variant & wl.PMASK_PAPER:   # the paper's annihilation mask: ANNI block 0 only (two planes ANDed + gate)
        lazy_d, eager_d = blocks_needed_generic(npd), (npd + 1) // 2
        lazy = fixed + raw + cmp_blk * lazy_d + (raw + PMASK_PER_BLOCK)
        eager = fixed + raw + cmp_blk * eager_d + (raw + PMASK_PER_BLOCK)
        lazy_blocks, eager_blocks = 2.0 + lazy_d, 2.0 + eager_d
        cmp_blocks, extra_alu = lazy_d, PMASK_PER_BLOCK
    else:
        lazy_dp = blocks_needed_generic(npd) + blocks_needed_generic(npp)
        eager_dp = (npd + 1) // 2 + (npp + 1) // 2
        lazy = fixed + raw + cmp_blk * lazy_dp
        eager = fixed + raw + cmp_blk * eager_dp
        lazy_blocks, eager_blocks = 1.0 + lazy_dp, 1.0 + eager_dp   # + the MISC block
        cmp_blocks, extra_alu = lazy_dp, 0.0
    # the lazy count by pipe (for the three-term bound of SURVEY.md 8(d)): wide multiplies (FMA-heavy pipe, 4 cycles
    # each), 32-bit IMADs of the generic signed-sum compare (FMA-heavy pipe, 2 cycles each), everything else on the ALU pipe
    wide = WIDE_FIXED + WIDE_PER_BLOCK * lazy_blocks
    imad = 0.5 * CMP_PER_BLOCK * cmp_blocks
    alu = lazy - wide - imad
    assert abs(alu - (alu_fixed + LOP_PER_BLOCK * lazy_blocks + 0.5 * CMP_PER_BLOCK * cmp_blocks + extra_alu)) < 1e-9
    return dict(lazy=lazy, eager=eager, lazy_blocks=lazy_blocks, eager_blocks=eager_blocks, fixed=fixed,
                per_block=cmp_blk, wide=wide, imad=imad, alu=alu)


def variant_name(v: int) -> str:
    return {wl.PCPD: "PCPD", wl.TCPD: "TCPD", wl.QCPD: "QCPD", wl.CPD: "CPD"}[v & 0xff] + ("+paper-pmask" if v & wl.PMASK_PAPER else "")


def load_peaks() -> dict:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


# --------------------------------------------------------------------------
class ClockSampler:
    """Samples SM clocks and throttle reasons DURING the timed region (NVML)."""

    def __init__(self, index: int):
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop = threading.Event()
        self._thr = None

    def start(self):
        try:
            import pynvml

            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self._nv = None
            return
        self._thr = threading.Thread(target=self._loop, daemon=True)
        self._thr.start()

    def _loop(self):
        nv = self._nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4),
        }
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(0.05)

    def stop(self) -> dict:
        self._stop.set()
        if self._thr:
            self._thr.join(timeout=2)
        s = sorted(self.samples)
        return dict(sm_mhz=(s[len(s) // 2] if s else None), sm_max_mhz=self.max_mhz, reasons=sorted(self.reasons),
                    samples=len(s))


# --------------------------------------------------------------------------
def oracle_sample_rate(cfg: wl.Config, L_sample: int, n_cols: int, sweeps: int = 1) -> tuple[float, float]:
    """Times the CPU oracle AS IT STANDS on `n_cols` word columns (one thread
    each; ctypes releases the GIL) of a ring of L_sample sites with the config's
    d, p, variant, seed and schedule.  Returns (updates/s, seconds)."""
    import oracle
    from concurrent.futures import ThreadPoolExecutor

    handles = []
    for w in range(n_cols):
        o = oracle.Oracle(L_sample, cfg.n_replicas, cfg.d, cfg.p, cfg.seed, cfg.variant, words=[w])
        o.init(cfg.init)
        handles.append(o)
    t0 = time.perf_counter()
    with ThreadPoolExecutor(n_cols) as ex:
        list(ex.map(lambda o: o.run(sweeps), handles))
    dt = time.perf_counter() - t0
    # the oracle's instrumentation: Philox blocks per attempt-word a lazy evaluation needs to decide all 64
    # lanes of both masks (+ the MISC block); deterministic for a seed, does not influence any result
    global LAST_ORACLE_LAZY_BLOCKS
    st = [o.stats() for o in handles]
    aw = sum(x["attempt_words"] for x in st)
    LAST_ORACLE_LAZY_BLOCKS = (1.0 + sum(x["blocks_needed_D"] + x["blocks_needed_P"] for x in st) / aw) if aw else None
    for o in handles:
        o.close()
    return L_sample * 64.0 * n_cols * sweeps / dt, dt


LAST_ORACLE_LAZY_BLOCKS = None


def reference_arm(args, cfg: wl.Config) -> None:
    """--impl reference: there is no reference implementation (paper only), so
    this arm times the ORACLE on the box's host cores on the same config,
    metric and unit; each step = one sweep of a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cores = max(1, min(os.cpu_count() or 1, cfg.W, 16))
    L_sample = min(cfg.L, 1 << 15)
    for _ in range(args.warmup):
        oracle_sample_rate(cfg, L_sample, cores, 1)
    t_total, units = 0.0, 0.0
    for _ in range(args.steps):
        rate, dt = oracle_sample_rate(cfg, L_sample, cores, 1)
        t_total += dt
        units += rate * dt
    value = units / t_total
    sample = (f"{cfg.name} parameters (d, p, variant, seed, schedule) on a ring of L = {L_sample} sites, "
              f"word columns 0..{cores - 1} of {cfg.W}, one sweep per step, one thread per column")
    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=1e3 * t_total / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="u8", data="synthetic", impl="reference",
                config=dict(workload=cfg.name, L=cfg.L, n_replicas=cfg.n_replicas, d=cfg.d, p=cfg.p,
                            variant=variant_name(cfg.variant), sample=sample),
                cpu_baseline=dict(value=value, unit=UNIT, cores=cores, kind="oracle", sample=sample),
                e2e=dict(value=value, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0),
                gpu_launches=0)
    print(json.dumps(line), flush=True)


# Microbenchmark kinds of the INT peak curve (include/pcpd.h, csrc/microbench.cu): (kind, wide, alu-pipe ops, 32-bit IMAD)
# per step, for the two pipe models of DESIGN.md section 6.
PEAK_CURVE = (("lop3", 0, 0, 1, 0), ("imad32", 2, 0, 0, 1), ("wide", 8, 1, 0, 0), ("imad_hi", 6, 1, 0, 0),
              ("lop3+imad32", 4, 0, 1, 1), ("wide+lop3", 1, 1, 1, 0), ("wide+2lop3", 9, 1, 2, 0), ("wide+3lop3", 5, 1, 3, 0),
              ("wide+4lop3", 10, 1, 4, 0), ("wide+imad32", 11, 1, 0, 1), ("iadd3", 12, 0, 1, 0),
              ("wide+lop3+2lop3_one_register", 13, 1, 3, 0), ("wide+lop3+2iadd3", 14, 1, 3, 0),
              ("2wide+5lop3+imad32", 15, 2, 5, 1))


def int_peak_curve(pk, sm_mhz: float) -> dict:
    """Measured rate of every mix, in lanes per clock per SM, beside what the two pipe models predict: `independent`
    = ALU pipe (2 cycles per warp-instruction) and FMA-heavy pipe (wide 4, IMAD 2) issue side by side, limited only
    by one instruction per cycle; `coupled` = a wide multiply also takes 2 cycles of the resource the ALU-pipe
    instructions use: max(4 W + 2 I, 2 (W + A), W + A + I) cycles per step."""
    out = {}
    for name, kind, W, A, I in PEAK_CURVE:
        rate = pk.microbench(kind, 2000) / 148 / (sm_mhz * 1e6)
        n = W + A + I
        indep = 32.0 * 4 * n / max(4 * W + 2 * I, 2 * A, n)
        coupled = 32.0 * 4 * n / max(4 * W + 2 * I, 2 * (W + A), n)
        out[name] = dict(kind=kind, lanes_per_clk_per_sm=round(rate, 2), model_independent=round(indep, 1),
                         model_coupled=round(coupled, 1))
    return out


def kernel_label(h) -> str:
    if h.split_launch_count() > 0:
        return "column_kernel (one block per tile column: producer warps + two half-word update warps)"
    return "sweep_warp_kernel" + (" (run-time specialised on T_d, T_p: csrc/jit.cu)" if h.jit_state() == 1
                                  else " (built-in generic-threshold kernel)")


def measure_resident(pk, torch, cfg: wl.Config, rank: int, steps: int, warmup: int, barrier, sampler=None) -> dict:
    """Device-resident timing of one config: `steps` steps of pcpd_run(SWEEPS_PER_STEP) + pcpd_density after `warmup`
    untimed ones (CUDA events on the launching stream), then the sweep launches alone and the density call alone."""
    h = pk.Pcpd(cfg.L, cfg.n_replicas, cfg.d, cfg.p, cfg.seed, cfg.variant, word_offset=rank * cfg.W)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    ev[0].record()
    h.init(cfg.init)
    ev[1].record()
    torch.cuda.synchronize()
    init_ms = ev[0].elapsed_time(ev[1])
    counts = np.empty(cfg.n_replicas, dtype=np.uint32)

    def step():
        h.run(SWEEPS_PER_STEP)
        h.density(counts)

    for _ in range(warmup):
        step()
    barrier()
    l0 = pk.launch_count()
    if sampler:
        sampler.start()
    ev[0].record()
    for _ in range(steps):
        step()
    ev[1].record()
    barrier()
    clocks = sampler.stop() if sampler else None
    launches = pk.launch_count() - l0
    t_ms = ev[0].elapsed_time(ev[1])
    # ---- dominant kernel alone: sweep launch durations ----
    n_k = max(4, min(40, steps * SWEEPS_PER_STEP))
    kev = [torch.cuda.Event(enable_timing=True) for _ in range(n_k + 1)]
    torch.cuda.synchronize()
    kev[0].record()
    for i in range(n_k):
        h.run(1)
        kev[i + 1].record()
    torch.cuda.synchronize()
    sweep_ms = sum(kev[i].elapsed_time(kev[i + 1]) for i in range(n_k)) / n_k
    ev[2].record()
    for _ in range(3):
        h.density(counts)
    ev[3].record()
    torch.cuda.synchronize()
    density_ms = ev[2].elapsed_time(ev[3]) / 3
    return dict(h=h, t_ms=t_ms, init_ms=init_ms, sweep_ms=sweep_ms, density_ms=density_ms, launches=launches, clocks=clocks)


def jit_expected(cfg: wl.Config) -> bool:
    """Handles with more than 768 tile columns run the run-time specialised kernel."""
    return (cfg.L // min(cfg.L, 2048)) * cfg.W > 768 and os.environ.get("PCPD_JIT", "1") != "0"


def ours_arm(args, cfg: wl.Config) -> None:
    import torch
    import torch.distributed as dist

    import paper_1301_6082_b200 as pk
    from paper_1301_6082_b200 import build

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device - the PCPD path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    peaks = load_peaks()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- timed region 1: device-resident (value); weak scaling: every rank owns a cfg-sized shard of word columns ----
    m = measure_resident(pk, torch, cfg, rank, args.steps, args.warmup, barrier, ClockSampler(local_rank))
    h, clocks, launches, sweep_ms, density_ms = m["h"], m["clocks"], m["launches"], m["sweep_ms"], m["density_ms"]
    if jit_expected(cfg) and h.jit_state() != 1:
        # a box without NVRTC would silently time the slower built-in kernel: fail loudly instead (PCPD_JIT=0 to allow)
        raise SystemExit(f"bench.py: {cfg.name} did not get the run-time specialised kernel (jit_state = {h.jit_state()}): "
                         f"{pk.jit_message()}; set PCPD_JIT=0 to time the built-in kernel on purpose")
    t_ms = torch.tensor([m["t_ms"]], device="cuda")
    if world > 1:
        dist.all_reduce(t_ms, op=dist.ReduceOp.MAX)
    t_ms = float(t_ms.item())
    units_per_step = float(cfg.L) * cfg.n_replicas * SWEEPS_PER_STEP * world
    value = units_per_step * args.steps / (t_ms * 1e-3)

    # ---- timed region 2: end to end through the C ABI with HOST buffers -----
    host_lat = torch.empty((cfg.L, cfg.W), dtype=torch.int64).pin_memory()
    host_cnt = torch.empty(cfg.n_replicas, dtype=torch.int32).pin_memory()
    h.get_lattice_ptr(host_lat.data_ptr())
    e2e_steps = max(2, min(args.steps, 5))
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]

    def e2e_step():
        # one call of the C ABI: H2D of the step's input lattice (cut into column chunks whose copies overlap the
        # sweeps of the chunks before), SWEEPS_PER_STEP sweeps, density, D2H of the counts
        h.step_from_host_ptr(host_lat.data_ptr(), SWEEPS_PER_STEP, host_cnt.data_ptr())

    def timed_e2e(fn):
        fn()
        barrier()
        t0 = time.perf_counter()
        ev[0].record()
        for _ in range(e2e_steps):
            fn()
        ev[1].record()
        barrier()
        wall = time.perf_counter() - t0
        e_ms = torch.tensor([max(ev[0].elapsed_time(ev[1]), 0.0)], device="cuda")
        if world > 1:
            dist.all_reduce(e_ms, op=dist.ReduceOp.MAX)
        return units_per_step * e2e_steps / (float(e_ms.item()) * 1e-3), wall

    e2e_canonical, _ = timed_e2e(e2e_step)
    # the same step from a host lattice kept in the device's own column-major order [w][i] (pcpd_step_from_host_columns:
    # contiguous chunk copies straight into the lattice, no staging, no transpose) - the faster of the two public calls
    host_cols = torch.empty((cfg.W, cfg.L), dtype=torch.int64).pin_memory()
    host_cols.numpy()[:] = host_lat.numpy().T
    del host_lat
    e2e_value, wall = timed_e2e(lambda: h.step_from_host_columns_ptr(host_cols.data_ptr(), SWEEPS_PER_STEP, host_cnt.data_ptr()))
    del host_cols

    if rank == 0:
        # INT roofline.  Nominal issue peak = 4 schedulers x 32 lanes per SM per clock.  The
        # kernel's instruction mix (IMAD.WIDE.U32 + ALU-pipe logic) cannot reach it: measured by the microbenchmark
        # curve below (run live here) every instruction of such a mix costs 2 issue cycles per scheduler, i.e. the
        # mix peaks at ~64 lanes/clk/SM.  `peak` is the highest measured rate over those mixes.
        nominal_peak = 148 * 128 * peaks["sm_max_mhz"] * 1e6
        curve = int_peak_curve(pk, peaks["sm_max_mhz"])
        to_rate = lambda name: curve[name]["lanes_per_clk_per_sm"] * 148 * peaks["sm_max_mhz"] * 1e6
        alu_peak, imad_peak, wide_peak = (to_rate(k) for k in ("lop3", "imad32", "wide"))
        # peak of the kernel's kind of mix (wide multiplies + logic): the HIGHEST rate any such mix reaches on the curve
        mix_names = ("wide+lop3", "wide+2lop3", "wide+3lop3", "wide+4lop3", "wide+lop3+2lop3_one_register",
                     "wide+lop3+2iadd3", "2wide+5lop3+imad32")
        mix_best = max(mix_names, key=to_rate)
        mix_peak = to_rate(mix_best)

        def int_roofline(c: wl.Config, launch_ms: float) -> dict:
            alg = algorithmic_instr_per_attempt_word(c)
            aw = float(c.L) * c.W                                   # attempt-words per sweep launch
            achieved = alg["lazy"] * aw / (launch_ms * 1e-3)
            # SURVEY.md 8(d)'s three-term bound with the measured per-pipe peaks (pipes assumed independent)
            t_three = aw * max(alg["lazy"] / nominal_peak, alg["alu"] / alu_peak, alg["wide"] / wide_peak + alg["imad"] / imad_peak)
            hbm = 2.0 * c.lattice_bytes / (launch_ms * 1e-3) / 1e9
            return dict(alg=alg, achieved=achieved, frac=achieved / mix_peak, frac_three_term=t_three / (launch_ms * 1e-3),
                        frac_eager=alg["eager"] * aw / (launch_ms * 1e-3) / mix_peak, frac_of_nominal_issue=achieved / nominal_peak,
                        hbm_gbs=hbm, hbm_frac=hbm / peaks["hbm_gbs"])

        r = int_roofline(cfg, sweep_ms)
        traffic = NCU_TRAFFIC_BYTES.get(cfg.name)
        roof = dict(bound="alu", achieved=r["achieved"] / 1e12, peak=mix_peak / 1e12, unit="Tinstr/s", frac=r["frac"],
                    frac_three_term=r["frac_three_term"],
                    traffic=traffic[0] if traffic else None,
                    traffic_source=(traffic[1] + " (constant from that ncu capture, not measured by this run)") if traffic else None,
                    kernel=kernel_label(h), launch_ms=sweep_ms,
                    instr_per_attempt_word=r["alg"]["lazy"], lazy_blocks=r["alg"]["lazy_blocks"],
                    instr_by_pipe=dict(wide=r["alg"]["wide"], imad32=r["alg"]["imad"], alu=r["alg"]["alu"]),
                    frac_eager=r["frac_eager"], frac_of_nominal_issue=r["frac_of_nominal_issue"],
                    peak_source="measured live: the highest rate over the pcpd_microbench mixes of IMAD.WIDE.U32 and logic "
                                f"(int_peak_curve: '{mix_best}', {mix_peak / 148 / (peaks['sm_max_mhz'] * 1e6):.1f} lanes/clk/SM; "
                                "profiles/r2_microbench.md shows why no such mix passes ~64); nominal issue peak "
                                f"148 SMs x 128 lanes/clk x {peaks['sm_max_mhz']:.0f} MHz = {nominal_peak / 1e12:.1f} Tinstr/s; "
                                "frac_three_term = max(N/issue, N_alu/alu_peak, N_wide/wide_peak + N_imad/imad_peak) with "
                                "the measured single-pipe peaks of int_peak_curve (pipes assumed independent)",
                    int_peak_curve=curve,
                    hbm=dict(achieved=r["hbm_gbs"], peak=peaks["hbm_gbs"], unit="GB/s", frac=r["hbm_frac"],
                             peak_source=peaks["source"]),
                    # the other kernel of the step: positional popcount, reads the lattice once (HBM-bound);
                    # density_ms includes the memset of the counts, their D2H copy and the stream synchronisation
                    density=dict(bound="hbm", achieved=cfg.lattice_bytes / (density_ms * 1e-3) / 1e9,
                                 peak=peaks["hbm_gbs"], unit="GB/s",
                                 frac=cfg.lattice_bytes / (density_ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                                 call_ms=density_ms))
        sched = h.schedule_info()
        h.close()
        # ---- the other BASELINE.json configs, a few steps each, same step and timing (north_star: "report
        # throughput on the synthetic configs"); N = 1 only ----
        configs = {cfg.name: dict(value=value, ms_per_step=t_ms / args.steps, sweep_ms=sweep_ms, frac=r["frac"],
                                  frac_three_term=r["frac_three_term"], hbm_frac=r["hbm_frac"], kernel=roof["kernel"])}
        if world == 1 and not args.no_other_configs:
            for other in wl.CONFIGS:
                if other.name == cfg.name:
                    continue
                mo = measure_resident(pk, torch, other, 0, 5, 3, barrier)
                ho = mo["h"]
                if jit_expected(other) and ho.jit_state() != 1:
                    raise SystemExit(f"bench.py: {other.name} did not get the run-time specialised kernel: {pk.jit_message()}")
                ro = int_roofline(other, mo["sweep_ms"])
                configs[other.name] = dict(value=float(other.L) * other.n_replicas * SWEEPS_PER_STEP * 5 / (mo["t_ms"] * 1e-3),
                                           ms_per_step=mo["t_ms"] / 5, sweep_ms=mo["sweep_ms"], frac=ro["frac"],
                                           frac_three_term=ro["frac_three_term"], hbm_frac=ro["hbm_frac"],
                                           kernel=kernel_label(ho), steps=5, warmup=3,
                                           l2="lattice larger than L2" if other.lattice_bytes > 200e6 else "lattice smaller than L2")
                ho.close()
        cores = max(1, min(os.cpu_count() or 1, cfg.W, 16))
        L_sample = min(cfg.L, 1 << 17)
        _, dt1 = oracle_sample_rate(cfg, L_sample, cores, 1)         # calibration sweep
        n_sw = int(max(1, min(200, round(15.0 / max(dt1, 1e-3)))))   # about 15 s of CPU work
        cpu_rate, cpu_dt = oracle_sample_rate(cfg, L_sample, cores, n_sw)
        sample = (f"{cfg.name} parameters on a ring of L = {L_sample} sites, word columns 0..{cores - 1} of {cfg.W}, "
                  f"{n_sw} sweeps, one thread per column ({cpu_dt:.1f} s)")
        line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup,
                    ms_per_step=t_ms / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None,
                    dtype="u64", data="synthetic",
                    config=dict(workload=cfg.name, L=cfg.L, n_replicas=cfg.n_replicas, d=cfg.d, p=cfg.p,
                                variant=variant_name(cfg.variant), seed=cfg.seed,
                                sweeps_per_step=SWEEPS_PER_STEP, step="pcpd_run(10) + pcpd_density",
                                schedule=sched, lattice_bytes=cfg.lattice_bytes,
                                l2="lattice (1 GiB at cfg4) is larger than L2; no flush needed" if cfg.lattice_bytes > 200e6
                                else "lattice smaller than L2 (correctness config)",
                                init_ms=m["init_ms"], density_ms=density_ms, parallelism=f"replica-word shards x{world}"),
                    roofline=roof, configs=configs,
                    cpu_baseline=dict(value=cpu_rate, unit=UNIT, cores=cores, kind="oracle", sample=sample,
                                      lazy_blocks_per_attempt_word=LAST_ORACLE_LAZY_BLOCKS),
                    e2e=dict(value=e2e_value, unit=UNIT, h2d_bytes_per_step=cfg.lattice_bytes,
                             d2h_bytes_per_step=4 * cfg.n_replicas, steps=e2e_steps, wall_s=wall,
                             call="pcpd_step_from_host_columns(pinned host lattice in column-major order [w][i], 10 sweeps, host counts)",
                             canonical_layout_value=e2e_canonical,
                             canonical_layout_call="pcpd_step_from_host(pinned host lattice in canonical order [i][w], 10 sweeps, "
                                                   "host counts): strided chunk copies + transpose"),
                    gpu_launches=int(launches), clocks=clocks)
        print(json.dumps(line), flush=True)
    else:
        h.close()
    if world > 1:
        dist.destroy_process_group()


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="cfg4", choices=sorted(wl.BY_NAME))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-other-configs", action="store_true", help="skip the short runs of the other BASELINE configs")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    cfg = wl.BY_NAME[args.config]
    if args.impl == "reference":
        reference_arm(args, cfg)
    else:
        ours_arm(args, cfg)


if __name__ == "__main__":
    main()
