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
  roofline   generation kernel only: algorithmic output bytes / its mean CUDA-event duration inside
             the timed steps, against MEASURED_PEAKS.json hbm_gbs; the fill-probe write peak of the
             same run is reported beside it
  cpu_baseline  the CPU oracle, as it stands, on all host cores, on a bounded sample of the workload

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


# Integer-bound generators (DESIGN.md 6.4/6.5): thread-instructions per number of the generation loop
# (SASS counts of the committed kernels, confirmed by ncu smsp__inst_executed in profiles/r01b_summary.md)
# against the issue peak 148 SMs x 4 schedulers x 32 lanes x sm_max_mhz.
ALU_INSTR_PER_NUMBER = {"gm19": 250, "gm29": 263, "gm31": 285, "gm61": 545, "gm55": 195, "gq58.1": 306,
                        "gq58.3": 148, "gq58.4": 103}


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
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": wall / max(1, args.steps) * 1e3,
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
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda") if need_flush else None
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

    # write peak of the same run (fill probe, same buffer)
    fill_ms = []
    for i in range(13):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        P.prand_fill_u32(out.data_ptr(), w.out_bytes // 4, 0x12345678)
        b.record()
        torch.cuda.synchronize()
        if i >= 3:
            fill_ms.append(a.elapsed_time(b))
    fill_gbs = w.out_bytes / (statistics.median(fill_ms) * 1e-3) / 1e9

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

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    peak, peak_src = load_peaks()
    k_ms = statistics.mean(kernel_ms)
    achieved = w.out_bytes / (k_ms * 1e-3) / 1e9
    traffic = load_traffic(last_kernel[0])
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "kernel": last_kernel[0], "kernel_ms": k_ms,
                "kernel_share_of_step": k_ms / ms_per_step,
                "algorithmic_bytes_per_launch": w.out_bytes, "peak_source": peak_src,
                "write_peak_same_run_gbs": fill_gbs, "frac_of_write_peak": achieved / fill_gbs}
    if w.gen in ALU_INSTR_PER_NUMBER:              # integer-bound: report against the issue peak
        ipn = ALU_INSTR_PER_NUMBER[w.gen]
        a_g = ipn * w.numbers / (k_ms * 1e-3) / 1e9
        p_g = alu_peak_ginstr()
        roofline = {"bound": "alu", "achieved": a_g, "peak": p_g, "unit": "Gthread-instr/s", "frac": a_g / p_g,
                    "traffic": traffic, "kernel": last_kernel[0], "kernel_ms": k_ms,
                    "kernel_share_of_step": k_ms / ms_per_step, "thread_instr_per_number": ipn,
                    "peak_source": "148 SMs x 4 schedulers x 32 lanes x sm_max_mhz (DESIGN.md 6.5)",
                    "out_gbs": achieved, "hbm_peak_gbs": peak}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": ARITH.get(w.gen, "u32/u64 modular"), "data": "synthetic",
        "config": config_of(w),
        "roofline": roofline,
        "e2e": e2e, "gpu_launches": launches, "clocks": clk.summary(),
    }
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
    peak, _ = load_peaks()
    names = args.sweep_workloads.split(",") if args.sweep_workloads else list(workloads.ALL)
    rows = []
    fill_buf = torch.empty(2 << 30, dtype=torch.uint8, device="cuda")
    fill_ms = []
    for i in range(13):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); P.prand_fill_u32(fill_buf.data_ptr(), fill_buf.numel() // 4, 1); b.record()
        torch.cuda.synchronize()
        if i >= 3:
            fill_ms.append(a.elapsed_time(b))
    fill_gbs = fill_buf.numel() / (statistics.median(fill_ms) * 1e-3) / 1e9
    del fill_buf
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    for name in names:
        w = workloads.ALL[name]
        tdt = {"u32": torch.int32, "f32": torch.float32, "f64": torch.float64}[w.dtype]
        gen_fn = {"u32": P.prand_generate_u32, "f32": P.prand_generate_f32, "f64": P.prand_generate_f64}[w.dtype]
        if w.seq:
            seq_name = "prand_generate_seq_" + w.dtype

            def gen_fn(h, ptr, n, _name=seq_name):
                P._generate(_name, h, ptr, n, None)
        out = torch.empty((w.n_per_stream, w.n_streams), dtype=tdt, device="cuda")
        init_ms = []
        h = None
        for i in range(3):
            if h:
                P.prand_free(h)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            h = P.prand_init(w.gen, w.seed, w.n_streams, w.block_len)
            torch.cuda.synchronize()
            init_ms.append((time.perf_counter() - t0) * 1e3)
        gen_ms = []
        for i in range(args.warmup + args.steps):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); gen_fn(h, out.data_ptr(), w.n_per_stream); b.record()
            torch.cuda.synchronize()
            if i >= args.warmup:
                gen_ms.append(a.elapsed_time(b))
        kernel = P.prand_last_kernel(h)
        P.prand_free(h)
        del out
        torch.cuda.empty_cache()
        med, best = statistics.median(gen_ms), min(gen_ms)
        gbs = w.out_bytes / (med * 1e-3) / 1e9
        row = {"workload": w.name, "gen": w.gen, "dtype": w.dtype, "n_streams": w.n_streams,
               "n_per_stream": w.n_per_stream, "kernel": kernel, "gen_ms_median": med, "gen_ms_best": best,
               "gnumbers_per_s": w.numbers / (med * 1e-3) / 1e9, "out_gbs": gbs, "frac_of_hbm_copy_peak": gbs / peak,
               "frac_of_write_peak": gbs / fill_gbs, "init_ms_best": min(init_ms),
               "init_streams_per_s": w.n_streams / (min(init_ms) * 1e-3)}
        rows.append(row)
        print(json.dumps(row), file=sys.stderr, flush=True)
    result = {"write_peak_gbs": fill_gbs, "hbm_copy_peak_gbs": peak, "rows": rows}
    with open(args.sweep, "w") as f:
        json.dump(result, f, indent=1)
    print(json.dumps({"sweep": args.sweep, "write_peak_gbs": fill_gbs, "n_rows": len(rows)}), flush=True)


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
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours" and not args.sweep:
        args.warmup = 3                          # timing rule: at least three warm-up steps
    w = workloads.ALL[args.workload]
    if args.sweep:
        return run_sweep(args)
    if args.impl == "reference":
        return run_reference(args, w)
    return run_ours(args, w)


if __name__ == "__main__":
    main()
