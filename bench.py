#!/usr/bin/env python
"""bench.py -- throughput of the PRAND hot path on B200 (BASELINE.json metric: Gnumbers/s).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C2] [--impl ours|reference]
                    [--sweep OUT.json]

One *step* = one pass of the whole hot path over one batch:
``prand_init`` (host operator preparation + stream-init kernel), ``prand_jump`` (all streams skip one
batch), ``prand_generate_<dtype>`` (recurrence + fused conversion + coalesced stores) and
``prand_free``.  The default workload is BASELINE.json ``configs[1]`` (C2: MRG32K3A, 65,536 streams,
block_len 2^76, 16,384 float64 per stream = 2^30 numbers, 8 GiB).  Prints ONE JSON line.

  value      whole-job Gnumbers/s, device-resident output, max over ranks of the CUDA-event time
  e2e        same metric through prand_generate_<dtype>_host (pinned HOST buffer; device->host copies
             and the operator-table uploads inside the timed region)
  roofline   generation kernel only: algorithmic bytes / its mean CUDA-event duration inside the timed steps,
             against the largest write-capable rate measured (MEASURED_PEAKS.json hbm_gbs, the fill probe and
             cudaMemsetAsync of the same run; the kernels only store, and stores alone beat the copy peak);
             frac_of_copy_peak keeps the MEASURED_PEAKS figure; roofline.per_config = one short row per
             configuration (kernel, ms, Gnumbers/s, bound, frac, instructions per number, oracle Gnumbers/s)
  cpu_baseline  the CPU oracle, as it stands, on all host cores, on a bounded sample of the workload

  per_config every other BASELINE.json configuration (C1, C3, C4 x2, C5 x9) and the paper's Table 7 task
             (T7 x2), generation call alone: gen_ms, Gnumbers/s, bound, frac, kernel, init_ms, clocks; plus
             launch_floor_us (empty kernel) and memset_write_peak_gbs (N = 1 only)

``--impl reference`` times the oracle alone (this tier's reference arm).  ``--gpus N`` under torchrun
shards the block-split family by stream index (weak scaling, no data-path collective).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads  # noqa: E402

METRIC = "Gnumbers/s per generator on 1 B200; % of measured HBM-write roofline"
UNIT = "Gnumbers/s"
ARITH = {"lfsr113": "u32", "mrg32k3a": "u32 (32x32->64 mul, mod 2^32-c) + f64 scale", "mt19937": "u32"}


# State bytes per stream: read once and written once per generate call.
STATE_BYTES = {"lfsr113": 16, "mrg32k3a": 24, "mt19937": 2496, "gm19": 256, "gm29": 256, "gm31": 256,
               "gm55": 128, "gm61": 512, "gq58.1": 512, "gq58.3": 192, "gq58.4": 128}
ALU_BOUND = {"gm19", "gm29", "gm31", "gm55", "gm61", "gq58.1", "gq58.3", "gq58.4"}
# SURVEY.md 8(d) table, "Algorithmic integer work / number (estimate)": the planning figure the ncu count of a kernel
# is read against (the alu `frac` is issue-slot utilisation of the kernel's OWN instruction count; it says how busy
# the SM is, and only together with count <= estimate how close the kernel is to the algorithm's cost)
SURVEY_INSTR_PER_NUMBER = {"gm19": "~290", "gm29": "~290", "gm31": "~320", "gm61": "650-800", "gm55": "~200",
                           "gq58.4": "~200", "gq58.3": "~300", "gq58.1": "300-800"}


def load_alu_counts():
    """Thread-instructions per number of the integer-bound generation kernels, as counted by ncu
    (smsp__inst_executed.sum x 32 / numbers) in the committed --set full captures: profiles/alu_counts.csv
    is written from those captures (its `source` column names the details file), never edited by hand; the pipe
    utilisations ncu measured in the same capture (ALU pipe, FMA-pipe cycles, issue slots) ride along."""
    import csv
    path = os.path.join(ROOT, "profiles", "alu_counts.csv")
    out = {}
    if os.path.exists(path):
        with open(path, newline="") as f:
            for row in csv.DictReader(f):
                pipes = {k: float(row[k]) for k in ("alu_pipe_pct", "fma_pipe_cycles_pct", "issue_active_pct", "fmaheavy_pipe_cycles_pct",
                                                   "fp64_pipe_pct") if row.get(k)}
                out[row["kernel"]] = (float(row["thread_instr_per_number"]), row["source"], pipes)
    return out


def algorithmic_bytes(w):
    """output element + state read and write-back amortised over n_per_stream; a
    single-sequence fill (T7) counts its output only."""
    if w.seq:
        return w.out_bytes
    return w.out_bytes + 2 * STATE_BYTES[w.gen] * w.n_streams


def alu_peak_ginstr():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    mhz = 1965.0
    if os.path.exists(path):
        with open(path) as f:
            mhz = float(json.load(f).get("sm_max_mhz", mhz))
    return 148 * 4 * 32 * mhz * 1e6 / 1e9


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def load_traffic(kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` from the committed
    ncu --set full capture (profiles/traffic.csv names the details file it came from), or None."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(path):
        return None
    import csv
    with open(path, newline="") as f:
        for row in csv.DictReader(f):
            if row["kernel"] == kernel:
                return int(row["dram_bytes_per_launch"])
    return None


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.002):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self._nv = None
        self._period = period_s

    def _run(self):
        nv = self._nv
        names = {
            nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
            nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
            nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake",
        }
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM))
                mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h)
                for bit, name in names.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(self._period)

    def __enter__(self):
        if self._nv is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        if self._thread:
            self._thread.join()

    def summary(self):
        return {"sm_mhz": statistics.median(self.samples) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ---- the CPU oracle as baseline / reference arm ----------------------------------------------------
def oracle_sample_rate(w, target_cpu_seconds: float, cores: int):
    """Time the oracle (as it stands) on a bounded sample of workload w: whole streams of the same
    block-split family, all rows, all host cores.  -> (Gnumbers/s, description)."""
    import oracle
    rows = min(w.n_per_stream, 16384)
    t0 = time.perf_counter()
    oracle.streams(w.gen, w.seed, 0, 2, w.block_len, rows, w.dtype, threads=1)     # calibration
    per_stream = max((time.perf_counter() - t0) / 2, 1e-6)
    n_streams = int(target_cpu_seconds / per_stream)
    n_streams = max(cores, min(w.n_streams, n_streams - n_streams % cores))
    t0 = time.perf_counter()
    oracle.streams(w.gen, w.seed, 0, n_streams, w.block_len, rows, w.dtype, threads=cores)
    dt = time.perf_counter() - t0
    sample = f"streams 0..{n_streams - 1} x {rows} rows of {w.name} ({n_streams * rows} numbers, {dt:.2f} s wall)"
    return n_streams * rows / dt / 1e9, sample


def run_reference(args, w):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    oracle.build()
    cores = os.cpu_count() or 1
    per_step_cpu_s = max(2.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_sample_rate(w, per_step_cpu_s, cores)
    rates, sample = [], ""
    t0 = time.perf_counter()
    for _ in range(args.steps):
        r, sample = oracle_sample_rate(w, per_step_cpu_s, cores)
        rates.append(r)
    wall = time.perf_counter() - t0
    value = statistics.mean(rates)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": wall / max(1, args.steps) * 1e3,      # measured: one step = one bounded sample of `config`
        "ms_per_step_extrapolated_full_config": w.numbers / (value * 1e9) * 1e3,   # all numbers of `config` at that rate
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": ARITH.get(w.gen, "u32/u64 modular"), "data": "synthetic",
        "config": config_of(w),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def config_of(w):
    return {"workload": f"{w.name}: {w.gen}, seed {w.seed}, {w.n_streams} streams, block_len 2^"
                        f"{w.block_len.bit_length() - 1}, {w.n_per_stream} {w.dtype} per stream, "
                        f"layout out[i*n_streams+s]",
            "numbers_per_step": w.numbers, "out_bytes_per_step": w.out_bytes,
            "step": "prand_init + prand_jump + prand_generate + prand_free",
            "l2": "output per step >> 126 MB L2 (no flush needed)" if w.out_bytes > (1 << 30)
                  else "L2 flushed between timed steps"}


# ---- our arm -----------------------------------------------------------------------------------------
def hbm_peak(peak, peak_src, fill_gbs=None, memset_gbs=None):
    """Denominator of the HBM rows.  The generation kernels only store, and a pure-store stream can run faster than
    the read+write copy MEASURED_PEAKS.json was taken with, so the peak is the LARGEST write-capable rate measured:
    MEASURED_PEAKS hbm_gbs, the fill probe of this run, cudaMemsetAsync of this run (SURVEY.md 8(d) "Write peak")."""
    cands = [(peak, peak_src)]
    if fill_gbs:
        cands.append((fill_gbs, "fill probe of this run (prand_fill_u32: one 128-bit st.global.cs per thread, CTAs in launch order)"))
    if memset_gbs:
        cands.append((memset_gbs, "cudaMemsetAsync of this run"))
    return max(cands, key=lambda c: c[0])


def roofline_of(w, kernel, k_ms, peak, peak_src, share=None, fill_gbs=None, memset_gbs=None):
    """The bench line's `roofline` object for one launch of `kernel` that took k_ms on workload w."""
    alg = algorithmic_bytes(w)
    out_gbs = w.out_bytes / (k_ms * 1e-3) / 1e9
    alg_gbs = alg / (k_ms * 1e-3) / 1e9
    traffic = load_traffic(kernel)
    wpeak, wsrc = hbm_peak(peak, peak_src, fill_gbs, memset_gbs)
    if w.gen in ALU_BOUND:                         # integer-bound: report against the issue peak
        counts = load_alu_counts()
        ipn, src, pipes = counts.get(kernel, (None, None, {}))
        p_g = alu_peak_ginstr()
        a_g = ipn * w.numbers / (k_ms * 1e-3) / 1e9 if ipn else None
        r = {"bound": "alu", "achieved": a_g, "peak": p_g, "unit": "Gthread-instr/s",
             "frac": a_g / p_g if a_g else None, "traffic": traffic, "kernel": kernel, "kernel_ms": k_ms,
             "thread_instr_per_number": ipn, "thread_instr_source": src, "ncu_pipe_pct": pipes,
             "survey_estimate_instr_per_number": SURVEY_INSTR_PER_NUMBER.get(w.gen),
             "frac_is": "issue-slot utilisation of the kernel's own ncu instruction count",
             "peak_source": "148 SMs x 4 schedulers x 32 lanes x sm_max_mhz (DESIGN.md 6.5, profiles/pipe_rates.md)",
             "out_gbs": out_gbs, "hbm_peak_gbs": wpeak, "frac_of_hbm": alg_gbs / wpeak}
    else:
        r = {"bound": "hbm", "achieved": alg_gbs, "peak": wpeak, "unit": "GB/s", "frac": alg_gbs / wpeak,
             "traffic": traffic, "kernel": kernel, "kernel_ms": k_ms,
             "algorithmic_bytes_per_launch": alg, "out_bytes_per_launch": w.out_bytes, "out_gbs": out_gbs,
             "peak_source": wsrc + " = the largest of the measured write-capable rates",
             "copy_peak_gbs": peak, "copy_peak_source": peak_src, "frac_of_copy_peak": alg_gbs / peak}
        if fill_gbs:
            r["write_peak_same_run_gbs"] = fill_gbs
            r["frac_of_write_peak"] = alg_gbs / fill_gbs
        if memset_gbs:
            r["memset_write_peak_gbs"] = memset_gbs
        # a kernel cannot beat the roofline: a fraction above 1 means the denominator is too low, not that the kernel is fast
        if r["frac"] > 1.0:
            raise SystemExit(f"bench.py: {w.name} {kernel}: {alg_gbs:.0f} GB/s exceeds the HBM peak {wpeak:.0f} GB/s "
                             f"({wsrc}): the roofline denominator is too low")
    if share is not None:
        r["kernel_share_of_step"] = share
    return r


def event_ms(torch, fn, n, warm=3, before=None):
    """CUDA-event durations (ms) of n calls of fn on torch's current stream, each after `before()`."""
    out = []
    for i in range(warm + n):
        if before:
            before()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); fn(); b.record()
        torch.cuda.synchronize()
        if i >= warm:
            out.append(a.elapsed_time(b))
    return out


def write_peaks(torch, P, nbytes=2 << 30):
    """Write roofline of this run: the fill probe (128-bit st.global.cs of a constant) and cudaMemsetAsync."""
    buf = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    fill = event_ms(torch, lambda: P.prand_fill_u32(buf.data_ptr(), nbytes // 4, 0x12345678), 10)
    mset = event_ms(torch, lambda: P.prand_probe_memset(buf.data_ptr(), 0x5A, nbytes), 10)
    del buf
    return nbytes / (statistics.median(fill) * 1e-3) / 1e9, nbytes / (statistics.median(mset) * 1e-3) / 1e9


def launch_floor_us(torch, P):
    """Empty kernel on the same stream: event-to-event time of one launch (what a small configuration's
    event pair measures at least), and the per-launch time of 1000 back-to-back launches."""
    single = event_ms(torch, P.prand_probe_empty, 200, warm=20)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    a.record()
    for _ in range(1000):
        P.prand_probe_empty()
    b.record()
    torch.cuda.synchronize()
    return {"single_event_pair_us_median": statistics.median(single) * 1e3,
            "single_event_pair_us_min": min(single) * 1e3,
            "back_to_back_us_per_launch": a.elapsed_time(b)}


def time_config(torch, P, w, steps, warmup, flush, peak, peak_src, device_index=0, fill_gbs=None, memset_gbs=None,
                cpu_seconds=0.0):
    """One per_config row: stream initialisation (wall clock around prand_init + synchronise, host
    operator preparation included) and the generation call alone (CUDA events, L2 flushed before each)."""
    tdt = {"u32": torch.int32, "f32": torch.float32, "f64": torch.float64}[w.dtype]
    name = ("prand_generate_seq_" if w.seq else "prand_generate_") + w.dtype
    out = torch.empty((w.n_per_stream, w.n_streams), dtype=tdt, device="cuda")
    init_ms, h = [], None
    for _ in range(3):
        if h:
            P.prand_free(h)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        h = P.prand_init(w.gen, w.seed, w.n_streams, w.block_len)
        torch.cuda.synchronize()
        init_ms.append((time.perf_counter() - t0) * 1e3)
    l0 = P.prand_launch_count()
    with ClockSampler(device_index) as clk:
        gen_ms = event_ms(torch, lambda: P._generate(name, h, out.data_ptr(), w.n_per_stream, None), steps,
                          warm=warmup, before=flush.zero_)
    launches = (P.prand_launch_count() - l0) // (steps + warmup)
    kernel = P.prand_last_kernel(h)
    P.prand_free(h)
    del out
    torch.cuda.empty_cache()
    med = statistics.median(gen_ms)
    roof = roofline_of(w, kernel, med, peak, peak_src, fill_gbs=fill_gbs, memset_gbs=memset_gbs)
    cpu = None
    if cpu_seconds > 0:                     # SURVEY.md 8(d) "Oracle timing": the oracle on this configuration, same run
        cores = os.cpu_count() or 1
        v, sample = oracle_sample_rate(w, cpu_seconds, cores)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
    return {"cpu_baseline": cpu, "hbm_peak_gbs": roof.get("hbm_peak_gbs", roof["peak"]),
            "survey_estimate_instr_per_number": roof.get("survey_estimate_instr_per_number"),
            "workload": w.name, "gen": w.gen, "dtype": w.dtype, "n_streams": w.n_streams,
            "n_per_stream": w.n_per_stream, "api": name, "kernel": kernel, "launches_per_call": launches,
            "gen_ms": med, "gen_ms_best": min(gen_ms), "gnumbers_per_s": w.numbers / (med * 1e-3) / 1e9,
            "bound": roof["bound"], "frac": roof["frac"], "out_gbs": roof["out_gbs"],
            "algorithmic_bytes": algorithmic_bytes(w), "frac_of_hbm": roof.get("frac_of_hbm", roof["frac"]),
            "thread_instr_per_number": roof.get("thread_instr_per_number"), "ncu_pipe_pct": roof.get("ncu_pipe_pct"),
            "init_ms": min(init_ms), "init_streams_per_s": w.n_streams / (min(init_ms) * 1e-3),
            "clocks": clk.summary()}


def jump_methods(torch, P):
    """the paper's own jump algorithms beside the library's default ones -- best wall time of
    prand_init + synchronise (3 runs) for 2^20 LFSR113 streams by the GF(2) matrix path and by the 128-table
    method, and of a prand_jump of 2^20 MT19937 steps on 512 streams from the device-resident
    polynomial table against host polynomial arithmetic with a cold cache."""
    def best(fn, reps=3):
        ts = []
        for _ in range(reps):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            fn()
            torch.cuda.synchronize()
            ts.append((time.perf_counter() - t0) * 1e3)
        return min(ts)

    out = {}
    w = workloads.ALL["C5-lfsr113"]
    for name, hook in (("matrix", None), ("table", "table")):
        P.prand_debug_set("PRAND_LFSR_INIT", hook)
        hs = []
        out[f"lfsr113_init_{w.n_streams}_streams_{name}_ms"] = best(
            lambda: hs.append(P.prand_init(w.gen, w.seed, w.n_streams, w.block_len)))
        for h in hs:
            P.prand_free(h)
    P.prand_debug_set("PRAND_LFSR_INIT", None)
    c3 = workloads.ALL["C3"]
    h = P.prand_init(c3.gen, c3.seed, c3.n_streams, c3.block_len)
    k = [0]

    def jump():
        k[0] += 1
        P.prand_jump(h, 1 << (20 + k[0]))             # a new tabulated distance every time: no cached ladder helps
    out["mt19937_jump_512_streams_table_ms"] = best(jump)
    P.prand_debug_set("PRAND_MT_POLY", "host")
    out["mt19937_jump_512_streams_host_polynomial_ms"] = best(jump)
    P.prand_debug_set("PRAND_MT_POLY", None)
    P.prand_free(h)
    return out


def device_api_rates(torch, P):
    """the device-callable API (include/prand_device.cuh) through the library's example kernels --
    one thread per stream calling next_u32() -- beside the bulk kernel on the same family (65,536 streams x 2048 u32;
    MT19937: one warp per stream, 2048 streams x 65,536), and stream initialisation by skip-ahead on the device
    (prand_device_api_init_fill: skipahead + 16 numbers per stream).  CUDA-event medians of 5 calls after 2 warm-ups."""
    out = {}
    for gen, seed, ns, L, n in (("lfsr113", 12345, 65536, 2**33, 2048), ("mrg32k3a", 12345, 65536, 2**76, 2048),
                                ("gm31", 1, 65536, 2**26, 2048), ("gq58.4", 1, 65536, 2**26, 2048),
                                ("mt19937", 5489, 2048, 2**64, 65536)):
        g = P.Generator(gen, seed, ns, L)
        bulk = statistics.median(event_ms(torch, lambda: g.generate(n, "u32"), 5, warm=2))
        dev = statistics.median(event_ms(torch, lambda: g.device_api_fill(n, "u32"), 5, warm=2))
        g.close()
        b = P.Generator(gen, seed, 1, 0)
        ini = statistics.median(event_ms(torch, lambda: b.device_api_init_fill(ns if gen != "mt19937" else 256, L, 16, "u32"), 5, warm=2))
        b.close()
        out[gen] = {"n_streams": ns, "n_per_stream": n, "bulk_gnumbers_per_s": ns * n / bulk / 1e6,
                    "device_api_gnumbers_per_s": ns * n / dev / 1e6,
                    "device_init_streams": ns if gen != "mt19937" else 256, "device_init_ms": ini}
    return out


def run_ours(args, w):
    import torch
    import paper_1307_5869_b200 as P

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        if world == 1 and args.gpus > 1:
            raise SystemExit("--gpus N > 1 must be launched with torch.distributed.run (one rank per GPU)")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    P.lib()                                        # fails loudly if libprand.so is missing
    tdt = {"u32": torch.int32, "f32": torch.float32, "f64": torch.float64}[w.dtype]
    gen_fn = {"u32": P.prand_generate_u32, "f32": P.prand_generate_f32, "f64": P.prand_generate_f64}[w.dtype]
    host_fn = {"u32": P.prand_generate_u32_host, "f32": P.prand_generate_f32_host,
               "f64": P.prand_generate_f64_host}[w.dtype]
    from paper_1307_5869_b200 import sharding
    first, _ = sharding.weak_shard(w.n_streams, rank)   # weak scaling: rank r holds streams [r ns, (r+1) ns)
    out = torch.empty((w.n_per_stream, w.n_streams), dtype=tdt, device="cuda")
    need_flush = w.out_bytes <= (1 << 30)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    last_kernel = [""]

    def step(ev=None):
        h = P.prand_init(w.gen, w.seed, w.n_streams, w.block_len, first_stream=first)
        P.prand_jump(h, w.n_per_stream)            # a2: every stream skips one batch
        if ev:
            ev[0].record()
        gen_fn(h, out.data_ptr(), w.n_per_stream)
        if ev:
            ev[1].record()
        last_kernel[0] = P.prand_last_kernel(h)
        P.prand_free(h)

    for _ in range(args.warmup):
        step()
    kev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    sev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    launches0 = P.prand_launch_count()
    with ClockSampler(local_rank) as clk:
        t_all0, t_all1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t_all0.record()
        for i in range(args.steps):
            if need_flush:
                flush.zero_()
            sev[i][0].record()
            step(kev[i])
            sev[i][1].record()
        t_all1.record()
        barrier()
    launches = P.prand_launch_count() - launches0
    if need_flush:
        elapsed_ms = sum(a.elapsed_time(b) for a, b in sev)      # flushes excluded
    else:
        elapsed_ms = t_all0.elapsed_time(t_all1)
    kernel_ms = [a.elapsed_time(b) for a, b in kev]
    elapsed_ms = sharding.max_over_ranks(elapsed_ms, device="cuda")
    ms_per_step = elapsed_ms / args.steps
    value = world * w.numbers / (ms_per_step * 1e-3) / 1e9

    # write peak of the same run: fill probe on the same buffer, cudaMemsetAsync as the second opinion
    fill_ms = event_ms(torch, lambda: P.prand_fill_u32(out.data_ptr(), w.out_bytes // 4, 0x12345678), 10)
    mset_ms = event_ms(torch, lambda: P.prand_probe_memset(out.data_ptr(), 0x5A, w.out_bytes), 10)
    fill_gbs = w.out_bytes / (statistics.median(fill_ms) * 1e-3) / 1e9
    memset_gbs = w.out_bytes / (statistics.median(mset_ms) * 1e-3) / 1e9

    # end to end through the host-delivery entry point
    e2e = None
    if not args.no_e2e:
        host = torch.empty((w.n_per_stream, w.n_streams), dtype=tdt, pin_memory=True)
        ke = max(1, min(args.steps, 3))

        def e2e_step():
            h = P.prand_init(w.gen, w.seed, w.n_streams, w.block_len, first_stream=first)
            P.prand_jump(h, w.n_per_stream)
            host_fn(h, host.data_ptr(), w.n_per_stream)
            P.prand_free(h)

        e2e_step()
        barrier()
        up0 = P.prand_uploaded_bytes()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        a.record()
        for _ in range(ke):
            e2e_step()
        b.record()
        barrier()
        wall_ms = (time.perf_counter() - t0) * 1e3
        ev_ms = max(a.elapsed_time(b), wall_ms)      # the call returns after the data arrived: both agree
        ev_ms = sharding.max_over_ranks(ev_ms, device="cuda")
        e2e = {"value": world * w.numbers * ke / (ev_ms * 1e-3) / 1e9, "unit": UNIT,
               "h2d_bytes_per_step": (P.prand_uploaded_bytes() - up0) // ke,
               "d2h_bytes_per_step": w.out_bytes, "steps": ke, "warmup": 1, "ms_per_step": ev_ms / ke,
               "api": f"prand_generate_{w.dtype}_host (pinned host buffer)"}
        del host
    del out

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    peak, peak_src = load_peaks()
    k_ms = statistics.mean(kernel_ms)
    roofline = roofline_of(w, last_kernel[0], k_ms, peak, peak_src, share=k_ms / ms_per_step, fill_gbs=fill_gbs,
                           memset_gbs=memset_gbs)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": ARITH.get(w.gen, "u32/u64 modular"), "data": "synthetic",
        "config": config_of(w),
        "roofline": roofline,
        "e2e": e2e, "gpu_launches": launches, "clocks": clk.summary(),
        "write_peak_gbs": fill_gbs, "memset_write_peak_gbs": memset_gbs,
    }
    if world == 1 and not args.no_per_config:
        # every other configuration of BASELINE.json (+ the paper's Table 7 task), generation call alone
        torch.cuda.empty_cache()
        line["launch_floor_us"] = launch_floor_us(torch, P)
        rows = []
        if not args.no_cpu:
            import oracle
            oracle.build()
        for name in workloads.ALL:
            rows.append(time_config(torch, P, workloads.ALL[name], args.config_steps, 3, flush, peak, peak_src,
                                    local_rank, fill_gbs=fill_gbs, memset_gbs=memset_gbs,
                                    cpu_seconds=0.0 if args.no_cpu else 2.0))
            print(json.dumps(rows[-1]), file=sys.stderr, flush=True)
        line["per_config"] = rows
        # the same table in short form inside `roofline` (one row per generator / configuration of BASELINE.json)
        roofline["per_config"] = {
            r["workload"]: {"kernel": r["kernel"], "ms": round(r["gen_ms"], 5), "gnps": round(r["gnumbers_per_s"], 2),
                            "bound": r["bound"], "frac": round(r["frac"], 4) if r["frac"] is not None else None,
                            "instr_per_number": r["thread_instr_per_number"],
                            "survey_instr_per_number": r["survey_estimate_instr_per_number"],
                            "init_ms": round(r["init_ms"], 3),
                            "cpu_gnps": round(r["cpu_baseline"]["value"], 4) if r["cpu_baseline"] else None}
            for r in rows}
        line["jump_methods"] = jump_methods(torch, P)
        line["pipe_rates"] = pipe_rates(torch, P, local_rank, calls=7)
        line["device_api"] = device_api_rates(torch, P)
        line["per_config_note"] = ("generation call alone (prand_generate_* / prand_generate_seq_*), CUDA-event median of "
                                   f"{args.config_steps} calls after 3 warm-ups, 256 MB written before each call (L2 flush); "
                                   "frac: hbm = algorithmic bytes (output + 2 x state) / gen_ms / the largest measured write-capable "
                                   "rate (MEASURED_PEAKS hbm_gbs, fill probe, cudaMemsetAsync of this run); "
                                   "alu = ncu thread-instructions per number (profiles/alu_counts.csv) x numbers / gen_ms / "
                                   "issue peak; init_ms = best wall time of prand_init + synchronise (3 runs); cpu_baseline = the oracle on "
                                   "a ~2 s sample of the same configuration, all host cores")
    if world == 1 and not args.no_cpu:
        import oracle
        oracle.build()
        cores = os.cpu_count() or 1
        v, sample = oracle_sample_rate(w, 10.0, cores)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


# ---- per-generator sweep (all BASELINE.json configs; a table for DESIGN.md / profiles) ---------------
def run_sweep(args):
    import torch
    import paper_1307_5869_b200 as P

    torch.cuda.set_device(0)
    peak, peak_src = load_peaks()
    names = args.sweep_workloads.split(",") if args.sweep_workloads else list(workloads.ALL)
    fill_gbs, memset_gbs = write_peaks(torch, P)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    rows = []
    for name in names:
        rows.append(time_config(torch, P, workloads.ALL[name], args.steps, args.warmup, flush, peak, peak_src,
                                fill_gbs=fill_gbs, memset_gbs=memset_gbs))
        print(json.dumps(rows[-1]), file=sys.stderr, flush=True)
    result = {"write_peak_gbs": fill_gbs, "memset_write_peak_gbs": memset_gbs, "hbm_copy_peak_gbs": peak,
              "launch_floor_us": launch_floor_us(torch, P), "rows": rows}
    with open(args.sweep, "w") as f:
        json.dump(result, f, indent=1)
    print(json.dumps({"sweep": args.sweep, "write_peak_gbs": fill_gbs, "n_rows": len(rows)}), flush=True)


# ---- instruction rates of the SM pipes (profiles/pipe_rates.md) ----------------------------------------
def pipe_rates(torch, P, device_index=0, calls=15):
    """Dependent-free instruction-rate probes (prand_probe_pipe): thread-level operations per clock per SM at the SM
    clock read while they run -- confirms the issue peak the alu rows are divided by."""
    sms = torch.cuda.get_device_properties(device_index).multi_processor_count
    rows = []
    for op, name in enumerate(P.prand_probe_pipe_names()):
        ops = [0]

        def fn(op=op):
            ops[0] = P.prand_probe_pipe(op, 2000)
        with ClockSampler(device_index, period_s=0.001) as clk:
            ms = event_ms(torch, fn, calls, warm=3)
        mhz = clk.summary()["sm_mhz"] or 1965.0
        med = statistics.median(ms)
        rows.append({"op": name, "ms": med, "thread_ops": ops[0], "sm_mhz": mhz,
                     "ops_per_clk_per_sm": ops[0] / (med * 1e-3) / (mhz * 1e6) / sms})
    return {"pipe_rates": rows, "sms": sms}


def run_pipe_rates(args):
    import torch
    import paper_1307_5869_b200 as P

    torch.cuda.set_device(0)
    print(json.dumps(pipe_rates(torch, P)), flush=True)


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--workload", default=workloads.HEADLINE.name, choices=sorted(workloads.ALL))
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-delivery (end-to-end) leg")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--sweep", default=None, metavar="OUT.json", help="time every workload, write a table")
    ap.add_argument("--sweep-workloads", default=None, help="comma-separated workload names for --sweep")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config table (all other configs)")
    ap.add_argument("--config-steps", type=int, default=20, help="timed calls per per_config row (SURVEY.md 8(d): >= 20)")
    ap.add_argument("--pipe-rates", action="store_true", help="print the SM pipe instruction rates (probe kernels)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours" and not args.sweep:
        args.warmup = 3                          # timing rule: at least three warm-up steps
    w = workloads.ALL[args.workload]
    if args.pipe_rates:
        return run_pipe_rates(args)
    if args.sweep:
        return run_sweep(args)
    if args.impl == "reference":
        return run_reference(args, w)
    return run_ours(args, w)


if __name__ == "__main__":
    main()
