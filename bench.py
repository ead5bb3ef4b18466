#!/usr/bin/env python
"""bench.py — throughput of the dedispersion + single-pulse-search hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload ska] [--impl ours|reference]

A *step* is one pass of the whole hot path (time binning -> dedispersion of every DM range -> row
statistics -> boxcar SNR / peaks / candidate compaction) over one chunk of synthetic filterbank data.
  value  DM-trial x samples / s with the chunk already resident in HBM (CUDA events on the compute stream).
  e2e    the same metric through aa_run_dedispersion(HOST pointer) ... aa_get_candidates: H2D of the chunk from pinned
         host memory and D2H of the candidate list inside the timed region.
  roofline  dominant kernel = K2 (k_dedisperse, one launch per DM range); bound "alu" (integer adds), see DESIGN.md.
  cpu_baseline  the oracle (oracle/, single-threaded C++) timed on a bounded sample of the same workload on this host.
N > 1 (torchrun): every rank runs the same step on its own chunk (replicas over time chunks, no collective on the data
path); value = outputs of all ranks / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "dm_trial_samples_per_s"
UNIT = "DM-trial*samples/s"
SM_COUNT = 148


K2_KERNELS = ("k_dedisperse", "k_scatter_exceptions")      # k_dedisperse also matches k_dedisperse_bits and k_dedisperse_naive


def csrc_digest() -> str:
    """sha256 over the kernel and host sources of the library (names and contents, sorted): what a tracked ncu capture is tied to.
    (The GPU box has no .git, so a commit id cannot be checked there; the sources can.)"""
    import hashlib
    h = hashlib.sha256()
    for f in sorted((ROOT / "paper_1912_07704_b200" / "csrc").iterdir()):
        if f.suffix in (".cu", ".cuh", ".cpp", ".h"):
            h.update(f.name.encode())
            h.update(f.read_bytes())
    return h.hexdigest()[:16]


def k2_dram_traffic(workload: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of the K2 launches of one step, from the tracked ncu capture
    profiles/k2_dram_traffic.json (which names the command, the commit and the source digest it was captured at).
    Returns (bytes or None, note); the note says STALE when the library sources have changed since the capture."""
    f = ROOT / "profiles" / "k2_dram_traffic.json"
    if not f.exists():
        return None, "no capture (profiles/k2_dram_traffic.json is missing)"
    rec = json.loads(f.read_text())
    e = rec.get("workloads", {}).get(workload)
    if not e:
        return None, f"no capture for workload {workload!r} in profiles/k2_dram_traffic.json"
    at = e.get("csrc_sha256", rec.get("csrc_sha256"))
    fresh = at is not None and at == csrc_digest()
    note = f"profiles/k2_dram_traffic.json (commit {e.get('commit', rec.get('commit'))}, {e.get('launches')} launches)"
    if not fresh:
        note += "; STALE: the library sources have changed since this capture (csrc digest %s then, %s now)" % (at, csrc_digest())
    return e["bytes_per_step"], note


def record_traffic(csv_path: str, workload: str, commit: str, command: str, steps: int = 1) -> None:
    """Write one workload's entry of profiles/k2_dram_traffic.json from an ncu --csv launch list that holds
    dram__bytes_read.sum and dram__bytes_write.sum of `steps` identical steps (python bench.py --record-traffic CSV --workload W
    --traffic-steps N --traffic-commit ID --traffic-command '...'). Sums the K2 launches (K2_KERNELS) and divides by the steps."""
    import csv
    rd = wr = 0
    ids = set()
    with open(csv_path, newline="") as fh:
        rows = [r for r in csv.reader(fh) if len(r) >= 15 and r[0].isdigit()]
    for r in rows:
        name, metric, val = r[4], r[12], int(float(r[14].replace(",", "")))
        if not any(k in name for k in K2_KERNELS):
            continue
        if metric == "dram__bytes_read.sum":
            rd += val; ids.add(r[0])
        elif metric == "dram__bytes_write.sum":
            wr += val; ids.add(r[0])
    assert ids, f"no K2 launch with DRAM metrics in {csv_path}"
    assert len(ids) % steps == 0, f"{len(ids)} K2 launches do not divide into {steps} steps"
    rd, wr, nl = rd // steps, wr // steps, len(ids) // steps
    f = ROOT / "profiles" / "k2_dram_traffic.json"
    rec = json.loads(f.read_text()) if f.exists() else {"workloads": {}}
    rec.setdefault("workloads", {})[workload] = {"bytes_per_step": rd + wr, "read": rd, "written": wr, "launches": nl,
                                                 "commit": commit, "csrc_sha256": csrc_digest(), "command": command,
                                                 "source": "profiles/" + Path(csv_path).name}
    f.write_text(json.dumps(rec, indent=1) + "\n")
    print(json.dumps(rec["workloads"][workload]))


INT_LANES_PER_SM_CLK = 128      # 64 ALU-pipe (IADD3) + 64 FMA-pipe (IMAD) lanes per SM per clock, DESIGN.md "Roofline"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="ska", help="tiny | mid | ska | lowf | stream (BASELINE.json configs 0..4), ska16 (ska as 16-bit samples); "
                    "stream = the 600 s chunked pipeline under a 40 GB budget, a step is the whole stream")
    ap.add_argument("--noise-sigma", type=float, default=None, help="override the workload's noise sigma (input counts); used to record how "
                    "the 16-bit offset forms degrade as the noise outgrows the byte window (not a BASELINE.json configuration)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--record-traffic", default=None, metavar="CSV", help="no GPU work: write this workload's entry of "
                    "profiles/k2_dram_traffic.json from an ncu --csv launch list of one step (see record_traffic)")
    ap.add_argument("--traffic-commit", default="uncommitted")
    ap.add_argument("--traffic-steps", type=int, default=1)
    ap.add_argument("--traffic-command", default="")
    ap.add_argument("--input", default="noise", choices=["noise", "uniform"], help="noise: the workload's recipe (Gaussian noise + pulses); "
                    "uniform: uniform random samples over the whole range - every offset form is exception-heavy, so the line records the "
                    "cost of the dense routes (uint16 kernels / global-memory kernel); not a BASELINE.json configuration")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--nsamp", type=int, default=0, help="shorten (or lengthen) the workload's observation to this many samples: "
                    "same band, DM plan and tiling, used for profiler captures of the large configurations; the line then "
                    "names the workload '<name>@<nsamp>' and is not a BASELINE.json configuration")
    return ap.parse_args()


def outputs_of(w, n_out):
    return sum(r[2] * (n_out // r[3]) for r in w.ranges)


# ------------------------------------------------------------------------------------------------ clocks sampler
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML every 100 ms while the timed region runs."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.mhz, self.reasons, self.max_mhz, self.power = index, False, [], set(), None, []
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap", nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake"}
        while not self.stop_flag:
            try:
                self.mhz.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
                bits = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for b, n in names.items():
                    if bits & b:
                        self.reasons.add(n)
            except Exception:
                pass
            time.sleep(0.1)

    def summary(self):
        return {"sm_mhz": float(np.median(self.mhz)) if self.mhz else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "power_w_max": max(self.power) if self.power else None,
                "samples": len(self.mhz)}


# ------------------------------------------------------------------------------------------------ oracle legs (CPU)
def oracle_sample(w, x, n_out, rows_per_range: int):
    """The oracle as it stands on a bounded sample: time binning of the whole chunk (step a2, done once per job) plus
    `rows_per_range` evenly spaced DM rows of every range over the full chunk, each row taken through dedispersion ->
    statistics -> boxcar SNR -> peaks. Work is exactly linear in the number of rows, so the whole-job time is
    t_bin + sum_r t_rows(r) * ndms_r / rows_r (SURVEY §8(d) "CPU baseline"). Returns (job outputs, job seconds
    extrapolated, seconds actually spent, text)."""
    import oracle
    k = oracle.delay_constants(w.freqs_mhz, w.tsamp_s)
    B = max(r[3] for r in w.ranges)
    L = (x.shape[1] // B) * B
    t_start = time.perf_counter()
    binned = {}
    for b in sorted({r[3] for r in w.ranges}):
        binned[b] = oracle.bin_time(x, 0, L // b, b)                # step a2
    t_job = time.perf_counter() - t_start
    for r, rng in enumerate(w.ranges):
        b, T = rng[3], n_out // rng[3]
        idx = list(range(rng[2])) if rows_per_range is None else \
            sorted({int(round(q * (rng[2] - 1) / max(1, rows_per_range - 1))) for q in range(rows_per_range)})
        t0 = time.perf_counter()
        for i in idx:
            D = oracle.dedisperse(binned[b], k, rng, i, i + 1, T)
            mu, sg, *_ = oracle.row_stats(D[0])
            S, wb = oracle.boxcar_snr(D[0], w.widths, mu, sg, prefix=True)
            oracle.find_peaks(S[None, :], w.threshold)
        t_job += (time.perf_counter() - t0) * rng[2] / len(idx)
    spent = time.perf_counter() - t_start
    what = (f"the WHOLE job: binning + every one of the {w.ndms_total} DM rows (dedispersion+SPS), nothing extrapolated" if rows_per_range is None else
            f"binning of the full chunk + {rows_per_range} evenly spaced DM row(s) of each of the {len(w.ranges)} ranges over "
            f"the full chunk (dedispersion+SPS), extrapolated linearly in rows to all {w.ndms_total} rows")
    return outputs_of(w, n_out), t_job, spent, what


def run_reference(args, w):
    """--impl reference: the oracle timed on the host cores, same metric/config; each step = a bounded sample."""
    import datagen
    import oracle
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    pl, dms, dl = w.pulses()
    x = datagen.generate(w.seed, w.nchans, w.nsamp, pl, dl, **w.gen_kw)
    k = oracle.delay_constants(w.freqs_mhz, w.tsamp_s)
    g = oracle.chunk_geometry(k, w.ranges, w.nsamp)
    rows = 1 if w.nchans * w.nsamp > (1 << 28) else 3
    for _ in range(min(args.warmup, 1)):
        oracle_sample(w, x, g["n_out"], rows)
    outs, secs, spent, what = 0, 0.0, 0.0, ""
    for _ in range(args.steps):
        o, s, sp, what = oracle_sample(w, x, g["n_out"], rows)
        outs += o
        secs += s
        spent += sp
    v = outs / secs
    # ms_per_step is what a step (= one bounded sample) really took, so that steps x ms_per_step is this run's wall time; value is the
    # whole-job throughput the sample extrapolates to (work is exactly linear in DM rows), job_ms_extrapolated the job time behind it
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": min(args.warmup, 1), "ms_per_step": 1e3 * spent / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int64", "job_ms_extrapolated": 1e3 * secs / args.steps, "data": "synthetic",
            "config": {"workload": w.name, "nchans": w.nchans, "nsamp": w.nsamp, "ndms": w.ndms_total,
                       "note": "each step is a bounded sample of the workload: " + what},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": what},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------ our arm (GPU)
def run_ours(args, w):
    import torch
    import torch.distributed as dist
    import datagen
    import paper_1912_07704_b200 as aa

    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    # synthetic chunk of this rank (replicas over time chunks: a different seed per rank), pinned for the e2e leg
    pl, dms, dl = w.pulses()
    esz = 2 if w.input_bits == 16 else 1
    xh = torch.empty((w.nchans, w.nsamp), dtype=torch.uint16 if esz == 2 else torch.uint8, pin_memory=True)
    x = xh.numpy()
    datagen.generate(w.seed + 1000003 * rank, w.nchans, w.nsamp, pl, dl, out=x, **w.gen_kw)
    if args.input == "uniform":
        rs = np.random.default_rng(w.seed + rank)
        for c0 in range(0, w.nchans, 256):
            x[c0:c0 + 256] = rs.integers(0, w.max_value + 1, size=x[c0:c0 + 256].shape, dtype=x.dtype)
    xd = xh.cuda(non_blocking=False)

    compute, copy = torch.cuda.Stream(), torch.cuda.Stream()
    plan = aa.Plan(w.freqs_mhz, w.tsamp_s, w.ranges, w.widths, w.threshold, input_bits=w.input_bits,
                   input_max=w.max_value if esz == 2 else 0)
    st = aa.Strategy(plan, w.nsamp, compute_stream=compute, copy_stream=copy, max_candidates=1 << 22)
    h, info = st.handle, st.info
    assert info["nchunks"] == 1, "the benchmark workload must fit one chunk"
    outputs = outputs_of(w, info["n_out"])
    adds = outputs * w.nchans
    in_bytes = w.nchans * info["chunk_len"] * esz

    def step_resident():
        aa.aa_strategy_reset(h)
        aa.aa_run_dedispersion_device(h, xd, xd.stride(0) * esz)
        aa.aa_run_sps(h)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step_resident()
    aa.aa_synchronize(h)
    ncand = len(aa.aa_get_candidates(h, allow_overflow=True))

    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    k2_ms, parts = [], []
    launches = 0
    for a, b in evs:
        a.record(compute)
        step_resident()
        b.record(compute)
        # per-kernel-class CUDA-event times of this step (recorded by the library on the compute stream); reading them
        # synchronises, which also separates the steps
        tm = aa.aa_get_last_timings(h)
        k2_ms.append(tm["dedisp_ms"])
        parts.append(tm)
        launches += aa.aa_get_launch_count(h)
    barrier()
    sampler.stop_flag = True
    sampler.join()
    total_ms = sum(a.elapsed_time(b) for a, b in evs)
    t = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms = float(t.item())
    value = outputs * world * args.steps / (total_ms * 1e-3)

    # e2e: host pointer in, candidate list out, through the public C-ABI calls
    e2e = None
    if not args.no_e2e:
        def step_e2e():
            aa.aa_strategy_reset(h)
            aa.aa_run_dedispersion(h, x, xh.stride(0) * esz)
            aa.aa_run_sps(h)
            return aa.aa_get_candidates(h, allow_overflow=True)
        step_e2e()
        barrier()
        t0 = time.perf_counter()
        d2h = 0
        for _ in range(args.steps):
            c = step_e2e()
            d2h += c.nbytes + 8
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        t = torch.tensor([dt], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e = {"value": outputs * world * args.steps / float(t.item()), "unit": UNIT,
               "h2d_bytes_per_step": int(in_bytes), "d2h_bytes_per_step": int(d2h // args.steps),
               "ms_per_step": 1e3 * float(t.item()) / args.steps, "timer": "host wall clock around the C-ABI calls, synchronised"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # roofline of the dominant kernel (K2, all ranges of one step = 5 launches): integer adds, bound "alu"
    iadd3, mixed, imad, mhz = aa.aa_measure_int_add_peak3(compute, 300)
    k2 = float(np.mean(k2_ms)) * 1e-3
    peak = SM_COUNT * INT_LANES_PER_SM_CLK * (sampler.max_mhz or 1965) * 1e6
    t_hbm = (in_bytes + 4 * outputs) / (json.loads((ROOT / "MEASURED_PEAKS.json").read_text())["hbm_gbs"] * 1e9) \
        if (ROOT / "MEASURED_PEAKS.json").exists() else (in_bytes + 4 * outputs) / 6.65e12
    traffic_key = w.name if args.input == "noise" else w.name + "+uniform-input"      # a capture belongs to one workload AND input recipe
    roofline = {"bound": "alu", "kernel": "k_dedisperse + k_dedisperse_bits + k_scatter_exceptions (K2), the launches of all DM ranges of one step",
                "achieved": adds / k2 / 1e12, "peak": peak / 1e12, "unit": "Tadd/s (algorithmic 32-bit integer adds)",
                "frac": adds / k2 / peak, "traffic": k2_dram_traffic(traffic_key)[0],
                "traffic_note": "dram__bytes_read.sum + dram__bytes_write.sum of the K2 launches of one step, one ncu capture: "
                                + str(k2_dram_traffic(traffic_key)[1]) + "; compulsory bytes are input once + D once",
                "peak_how": f"derived: {SM_COUNT} SMs x {INT_LANES_PER_SM_CLK} integer-add lanes/clk (64 IADD3 + 64 IMAD) x max SM clock",
                "measured_iadd3_only_tadd_s": iadd3 / 1e12, "measured_iadd3_imad_mixed_tadd_s": mixed / 1e12, "measured_imad_only_tadd_s": imad / 1e12,
                "frac_of_measured_mixed": adds / k2 / max(mixed, iadd3), "frac_of_measured_iadd3_only": adds / k2 / iadd3,
                "microbench_sm_mhz": mhz, "k2_ms_per_step": k2 * 1e3, "t_hbm_compulsory_ms": t_hbm * 1e3,
                "algorithmic_adds_per_step": adds}
    mean = lambda key: float(np.mean([p[key] for p in parts]))
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "int32", "data": "synthetic",
            "config": {"workload": w.name if args.input == "noise" else w.name + "+uniform-input", "nchans": w.nchans, "nsamp": w.nsamp,
                       "tsamp_us": w.tsamp_s * 1e6, "ndms": w.ndms_total, "input_bits": w.input_bits, "input_max": w.max_value,
                       "ranges": [list(r) for r in w.ranges], "widths": list(w.widths), "threshold": w.threshold,
                       "outputs_per_step": outputs, "l2": "inputs larger than L2 (chunk %.2f GB in, %.2f GB out)" % (in_bytes / 1e9, 4 * outputs / 1e9),
                       "parallelism": "replicas over time chunks" if world > 1 else "single GPU"},
            "realtime_factor": (info["n_out"] * w.tsamp_s) / (total_ms * 1e-3 / args.steps),
            "realtime_factor_e2e": (info["n_out"] * w.tsamp_s) / (e2e["ms_per_step"] * 1e-3) if e2e else None,
            "breakdown_ms": {"bin_and_shift": mean("bin_ms"), "dedispersion": mean("dedisp_ms"), "row_stats": mean("stats_ms"),
                             "sps_peaks": mean("peaks_ms")},
            "candidates_per_step": ncand, "clocks": sampler.summary(), "e2e": e2e, "gpu_launches": int(launches),
            "roofline": roofline}
    if not args.no_cpu_baseline and world == 1:
        # Tiny and Mid: the whole oracle (seconds / a few minutes; SURVEY §8(d) "CPU baseline"); the large configurations: first,
        # middle and last DM row of every range
        rows = None if w.name.split("+")[0].split("@")[0] in ("tiny", "mid") and not args.nsamp else 3
        o, secs, spent, what = oracle_sample(w, x, info["n_out"], rows)
        line["cpu_baseline"] = {"value": o / secs, "unit": UNIT, "cores": 1, "kind": "oracle, full" if rows is None else "oracle", "sample": what,
                                "sample_seconds": spent, "host_cores_available": os.cpu_count()}
    print(json.dumps(line), flush=True)
    st.close()
    plan.close()
    if world > 1:
        dist.destroy_process_group()


def run_stream(args, w):
    """BASELINE.json configs[4]: the whole observation stays in pinned HOST memory; the strategy splits it into
    overlapping chunks under the budget; H2D of chunk n+1 is double-buffered over dedispersion+SPS of chunk n.
    A step = the whole stream. `value` = units / sum of the per-chunk kernel times (CUDA events, chunk resident);
    `e2e` = units / wall clock of the overlapped run loop (host pointer in, candidate list out)."""
    import torch
    import datagen
    import paper_1912_07704_b200 as aa
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    assert int(os.environ.get("WORLD_SIZE", "1")) == 1, "the stream workload is a single-GPU configuration (BASELINE.json)"
    torch.cuda.set_device(0)
    pl, dms, dl = w.pulses()
    t0 = time.perf_counter()
    xh = torch.empty((w.nchans, w.nsamp), dtype=torch.uint8, pin_memory=True)
    x = xh.numpy()
    datagen.generate(w.seed, w.nchans, w.nsamp, pl, dl, out=x)
    gen_s = time.perf_counter() - t0
    compute, copy = torch.cuda.Stream(), torch.cuda.Stream()
    plan = aa.Plan(w.freqs_mhz, w.tsamp_s, w.ranges, w.widths, w.threshold)
    st = aa.Strategy(plan, w.nsamp, budget_bytes=w.budget_bytes, compute_stream=compute, copy_stream=copy, max_candidates=1 << 23)
    h, info = st.handle, st.info
    chunks = [aa.aa_strategy_get_chunk(h, j) for j in range(info["nchunks"])]
    outputs = sum(outputs_of(w, c[2]) for c in chunks)

    def pass_timed():                       # kernels only: reading the timings synchronises after every chunk
        aa.aa_strategy_reset(h)
        ms = {"bin_ms": 0.0, "dedisp_ms": 0.0, "stats_ms": 0.0, "peaks_ms": 0.0}
        n = 0
        while True:
            aa.aa_run_dedispersion(h, x, xh.stride(0))
            status = aa.aa_run_sps(h)
            tm = aa.aa_get_last_timings(h)
            for k in ms:
                ms[k] += tm[k]
            n = aa.aa_get_launch_count(h)
            if status == aa.AA_STATUS_FINISHED:
                return ms, n

    def pass_e2e():
        aa.aa_strategy_reset(h)
        t = time.perf_counter()
        c = st.run(x)
        torch.cuda.synchronize()
        return time.perf_counter() - t, c

    for _ in range(min(args.warmup, 1)):
        pass_e2e()
    sampler = ClockSampler(0)
    sampler.start()
    kern, launches, e2e_s, ncand, d2h = [], 0, [], 0, 0
    for _ in range(args.steps):
        ms, n = pass_timed()
        kern.append(ms)
        launches += n
        dt, c = pass_e2e()
        e2e_s.append(dt)
        ncand, d2h = len(c), c.nbytes + 8 * len(chunks)
    sampler.stop_flag = True
    sampler.join()
    mean = lambda key: float(np.mean([k[key] for k in kern]))
    step_ms = mean("bin_ms") + mean("dedisp_ms") + mean("stats_ms") + mean("peaks_ms")
    adds = outputs * w.nchans
    k2 = mean("dedisp_ms") * 1e-3
    peak = SM_COUNT * INT_LANES_PER_SM_CLK * (sampler.max_mhz or 1965) * 1e6
    e2e_mean = float(np.mean(e2e_s))
    duration = w.nsamp * w.tsamp_s
    line = {"metric": METRIC, "value": outputs / (step_ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
            "warmup": min(args.warmup, 1), "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "int32", "data": "synthetic",
            "config": {"workload": w.name, "nchans": w.nchans, "nsamp": w.nsamp, "tsamp_us": w.tsamp_s * 1e6, "ndms": w.ndms_total,
                       "budget_bytes": w.budget_bytes, "chunk_len": info["chunk_len"], "overlap": info["overlap"],
                       "nchunks": info["nchunks"], "arena_bytes": info["arena_bytes_used"], "outputs_per_step": outputs,
                       "l2": "inputs larger than L2 (each chunk %.2f GB in)" % (w.nchans * info["chunk_len"] / 1e9),
                       "parallelism": "single GPU, double-buffered H2D", "host_generation_s": gen_s},
            "realtime_factor": duration / (step_ms * 1e-3), "realtime_factor_e2e": duration / e2e_mean,
            "breakdown_ms": {"bin_and_shift": mean("bin_ms"), "dedispersion": mean("dedisp_ms"), "row_stats": mean("stats_ms"),
                             "sps_peaks": mean("peaks_ms")},
            "candidates_per_step": ncand, "clocks": sampler.summary(),
            "e2e": {"value": outputs / e2e_mean, "unit": UNIT, "h2d_bytes_per_step": int(sum(w.nchans * c[1] for c in chunks)),
                    "d2h_bytes_per_step": int(d2h), "ms_per_step": 1e3 * e2e_mean,
                    "timer": "host wall clock around the run loop (aa_run_dedispersion(host) / aa_run_sps per chunk, aa_get_candidates)"},
            "gpu_launches": int(launches),
            "roofline": {"bound": "alu", "kernel": "k_dedisperse (K2), all ranges of all chunks", "achieved": adds / k2 / 1e12,
                         "peak": peak / 1e12, "unit": "Tadd/s (algorithmic 32-bit integer adds)", "frac": adds / k2 / peak,
                         "traffic": None, "k2_ms_per_step": k2 * 1e3, "algorithmic_adds_per_step": adds}}
    print(json.dumps(line), flush=True)
    st.close()
    plan.close()


def spawn_ranks(n: int) -> int:
    """Re-run this command as n ranks under torch.distributed.run on 127.0.0.1 (one process per GPU). Returns the exit code;
    refuses, with the reason, when the node shows fewer than n CUDA devices."""
    import socket
    import subprocess
    import torch
    have = torch.cuda.device_count() if torch.cuda.is_available() else 0
    if have < n:
        print(f"bench.py: --gpus {n} needs {n} CUDA devices on this node, {have} visible; not running (a line with n_gpus: {have} "
              f"would not be the measurement asked for)", file=sys.stderr)
        return 2
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), str(Path(__file__).resolve()), *sys.argv[1:]]
    return subprocess.call(cmd)


def main():
    args = parse()
    if args.record_traffic:
        record_traffic(args.record_traffic, args.workload, args.traffic_commit, args.traffic_command, args.traffic_steps)
        return
    launched = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        pass                                   # CPU arm: rank 0 runs, the others exit; no GPU count to check
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # started as plain `python bench.py --gpus N`: become N ranks (one process per GPU) the way the driver starts them,
        # or say why not. Never print an n_gpus: 1 line for a --gpus N request.
        sys.exit(spawn_ranks(args.gpus))
    elif args.gpus != launched:
        sys.exit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE = {launched}: start N ranks with --nproc-per-node N (or run "
                 f"`python bench.py --gpus N` and let it spawn them)")
    import datagen
    w = datagen.get_workload(args.workload)
    if args.nsamp:
        w = datagen.scaled(w, nsamp=args.nsamp, name=f"{w.name}@{args.nsamp}")
    if args.noise_sigma is not None:
        w = datagen.scaled(w, noise_sigma=args.noise_sigma, name=f"{w.name}+sigma{args.noise_sigma:g}")
    if args.impl == "reference":
        run_reference(args, w)
    elif w.budget_bytes:
        run_stream(args, w)
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()
