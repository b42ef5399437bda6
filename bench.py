#!/usr/bin/env python
"""bench.py -- LLOID hot-path throughput and latency on B200 (driver contract).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config N] [--precision split]

A STEP is one lloid_stream_push of one buffer of every detector against every bank of the workload:
a1 decimate -> a2 basis correlation -> a4 upsample -> a3 reconstruction -> a5 peaks.  The metric is BASELINE.json's:
template*detector*data-seconds filtered per wall-second (plus per-buffer latency).

With no --config the HEADLINE is the largest single-GPU workload, BASELINE.json configs[4] (full-scale: 1000 SVD banks x
1000 templates, 3 detectors, 1 s buffers), and the same JSON line carries the records of configs[1], [2] and [3]
(small-bank, mid-scale, low-latency 1/16 s buffers with p50/p99) under "other_configs".  `--config N` runs that config
alone.  `--gpus N` (N > 1) re-executes itself under torch.distributed.run with N ranks unless it is already running
under one; every rank filters an independent replica of the workload (weak scaling, no data-path collective).
Prints ONE JSON line on rank 0.  `--impl reference` times the float64 CPU oracle (oracle/) on the host cores.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "template*detector*data-seconds filtered per wall-second"
UNIT = "template*detector*data-s/s"
PREC = {"ffma": 0, "f16": 1, "split": 2}
PREC_DTYPE = {"ffma": "f32", "f16": "f16 operands, f32 accumulate", "split": "f16 product + fp8 (e4m3 x e5m2) hi/lo correction MMA, f32 accumulate"}
HEADLINE_CONFIG = 5                  # BASELINE.json configs[4]: the largest single-GPU workload
NESTED_CONFIGS = (2, 3, 4)           # carried inside the headline line


def parse(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=0,
                    help="BASELINE.json config number (1-based); default: headline config 5 with configs 2-4 nested")
    ap.add_argument("--precision", default=os.environ.get("LLOID_BENCH_PRECISION", "split"), choices=list(PREC))
    ap.add_argument("--banks", type=int, default=0, help="debug: use only the first n banks (0 = all; marks the run as reduced)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-nested", action="store_true", help="headline config only")
    ap.add_argument("--no-flush", action="store_true", help="keep L2 warm between steps (reported in config)")
    ap.add_argument("--plumbing-check", action="store_true",
                    help="exercise launcher -> ranks -> process group -> max-over-ranks -> rank-0 line over gloo, no filtering (CPU test)")
    return ap.parse_args(argv)


# ---------------------------------------------------------------------------------------------------------
# workload: which banks are chirp-SVD banks, which are shape-faithful stand-ins
# ---------------------------------------------------------------------------------------------------------
N_REAL_BANKS = 4        # evenly spaced chirp-SVD banks in the many-bank configs
N_INJ_BANKS = 4         # plus the banks hit by the first injections of the parity stream (tests/test_gpu_fullsize.py)


def parity_seconds(c):
    """Length of the live-history parity stream of a config: the longest template plus 2 s."""
    return int(c.T_max) + 2


def real_bank_ids(c, nb):
    """Banks built as real chirp-SVD banks: all of them for few-bank configs, else N_REAL_BANKS evenly spaced ones plus
    the banks of the first N_INJ_BANKS distinct injected banks of the config's seeded parity-stream injections."""
    if nb <= 8:
        return list(range(nb))
    ids = set(int(round(i * (nb - 1) / (N_REAL_BANKS - 1))) for i in range(N_REAL_BANKS))
    extra = []
    for inj in c.injections(parity_seconds(c)):
        if inj.bank < nb and inj.bank not in ids and inj.bank not in extra:
            extra.append(inj.bank)
        if len(extra) >= N_INJ_BANKS:
            break
    return sorted(ids | set(extra))


def bank_plan(cfg_no, n_banks_limit=0):
    """(config, list of bank descriptions).  Every bank keeps its REAL slice layout (rates, taps, delays from its own
    chirp masses); the banks of real_bank_ids are chirp-SVD banks, the others take the basis counts L^s of the nearest
    real bank, with seeded random orthonormal U and random R (SURVEY.md section 8d "scale handling")."""
    from workloads import CONFIGS
    c = CONFIGS[cfg_no]
    nb = c.n_banks if not n_banks_limit else min(n_banks_limit, c.n_banks)
    real = real_bank_ids(c, nb)
    return c, [("real", b) if b in real else ("standin", b, min(real, key=lambda r: (abs(r - b), r))) for b in range(nb)]


def real_banks(cfg_no, ids, info=None):
    """{bank index: chirp-SVD bank, float32-rounded}: workloads/bank_cache.py (parallel worker processes, .npz cache)."""
    from workloads.bank_cache import real_banks as _rb
    return _rb(cfg_no, ids, info)


def standin_bank(c, b, like, mcs=None):
    from workloads import random_bank
    T, lay = c.layout(b, c.mchirps() if mcs is None else mcs)
    Ls = [s.n_basis for s in like.slices]
    shape = [(rate, (e - s0) // (c.f0 // rate), Ls[min(i, len(Ls) - 1)]) for i, (rate, s0, e) in enumerate(lay)]
    return random_bank(c.seed(b), c.M, shape, f0=c.f0).as_f32()


def iter_banks(cfg_no, plan, describe=None, info=None, real=None):
    """Yield the planned banks one at a time (the caller uploads each and drops it)."""
    from workloads import CONFIGS
    c = CONFIGS[cfg_no]
    mcs = c.mchirps()
    if real is None:
        real = real_banks(cfg_no, [p[1] for p in plan if p[0] == "real"], info)
    for p in plan:
        bank = real[p[1]] if p[0] == "real" else standin_bank(c, p[1], real[p[2]], mcs)
        if describe is not None:
            describe.append(("real " if p[0] == "real" else "standin ") + bank.describe())
        yield bank


def build_workload(cfg_no, n_banks_limit, seconds, rank=0, only_real=True):
    """Banks (float32-rounded) and [n_det][seconds*f0] strain, seeded.  only_real: for the
    many-bank configs return just the real chirp-SVD banks (what the oracle legs sample)."""
    from workloads import make_strain
    c, plan = bank_plan(cfg_no, n_banks_limit)
    if only_real:
        plan = [p for p in plan if p[0] == "real"]
    banks = list(iter_banks(cfg_no, plan))
    # white N(0,1) strain per detector; ranks > 0 (weak scaling replicas) shift the detector seeds
    strain = np.stack([make_strain(c.seed(det) + 100 * rank, seconds * c.f0) for det in range(c.n_det)])
    return c, banks, strain


def config_dict(cfg_no, c, plan, reduced=False):
    """The `config` object of the JSON line: names the WORKLOAD only, identical for both arms (--impl ours / reference)."""
    n_real = sum(p[0] == "real" for p in plan)
    return {"workload": f"BASELINE.json configs[{cfg_no - 1}] ({c.name})" + (" REDUCED (--banks)" if reduced else ""),
            "n_banks": len(plan), "templates_per_bank": c.M, "n_detectors": c.n_det, "buffer_len": c.buffer_len,
            "banks": (f"{n_real} chirp-SVD banks + {len(plan) - n_real} shape-faithful stand-ins (real slice layout, L^s of the "
                      "nearest SVD bank, random orthonormal U / random R)")}


def max_over_ranks(t_local, device, world):
    """Timed-region seconds of the slowest rank (all_reduce MAX over the job's process group)."""
    if world <= 1:
        return float(t_local)
    import torch
    import torch.distributed as dist
    t = torch.tensor([t_local], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world, units_per_step_per_rank, steps, seconds):
    """Aggregate throughput of `world` independent replicas (weak scaling, no data-path collective)."""
    return world * units_per_step_per_rank * steps / seconds


def launcher_command(n, argv, port=None):
    """The command `--gpus N` re-executes: one rank per GPU of this node under torch.distributed.run."""
    port = port or os.environ.get("MASTER_PORT") or str(29500 + os.getpid() % 2000)
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(n), "--master-addr", "127.0.0.1",
            "--master-port", str(port), os.path.abspath(__file__)] + list(argv)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                                          "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.t.join(timeout=2)
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) >= 7 and r[3 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


# ---------------------------------------------------------------------------------------------------------
# the oracle legs (cpu_baseline and --impl reference): float64 numpy on the host cores, as it stands
# ---------------------------------------------------------------------------------------------------------
def oracle_step(banks, strain, k_hi, B):
    """One step's worth of oracle work: SNR of every bank x detector over the buffer ending at k_hi + peaks."""
    from oracle import find_peaks, lloid_snr
    for det in range(strain.shape[0]):
        dec = {}
        for bank in banks:
            rho = lloid_snr(bank, strain[det][:k_hi], k_hi - B, k_hi, decimated=dec)
            find_peaks(rho, B)


def blas_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads") for p in threadpool_info() if p.get("user_api") == "blas"]
        return max(n) if n else os.cpu_count()
    except Exception:
        return os.cpu_count()


def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.lower().startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def time_oracle(banks, strain, B, f0, budget_s, steps=5, warmup=0, n_total_banks=None):
    """Time `steps` oracle steps on a bounded sample: as many leading banks as fit ~budget_s per step."""
    n_det = strain.shape[0]
    hist = strain.shape[1] - (steps + warmup) * B
    assert hist >= 0
    t0 = time.perf_counter()
    oracle_step(banks[:1], strain, hist + B, B)                                  # calibration (untimed)
    t1 = time.perf_counter() - t0
    nb = int(max(1, min(len(banks), budget_s / max(t1, 1e-3))))
    sub = banks[:nb]
    for w in range(warmup):
        oracle_step(sub, strain, hist + (w + 1) * B, B)
    t0 = time.perf_counter()
    for s in range(steps):
        oracle_step(sub, strain, hist + (warmup + s + 1) * B, B)
    dt = time.perf_counter() - t0
    units = sum(b.M for b in sub) * n_det * (B / f0) * steps
    n_all = n_total_banks if n_total_banks is not None else len(banks)
    sample = (f"{nb} chirp-SVD bank(s) of the workload's {n_all} x {n_det} detectors x {steps} buffer(s) of {B} samples, float64 numpy"
              + ("; EXTRAPOLATED linearly in banks to the whole workload (rate per template*detector*data-second)" if nb < n_all else ""))
    return units / dt, dt / steps, sample


def cpu_baseline_record(value, sample):
    return {"value": value, "unit": UNIT, "cores": blas_threads(), "kind": "oracle", "sample": sample,
            "os_cpu_count": os.cpu_count(), "blas_threads": blas_threads(), "cpu_model": cpu_model()}


def run_reference(args):
    """--impl reference: the oracle as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    cfg_no = args.config or HEADLINE_CONFIG
    hist_s = 4
    c, plan = bank_plan(cfg_no, args.banks)
    _, banks, strain = build_workload(cfg_no, args.banks, hist_s + -(-(args.steps + args.warmup) * c.buffer_len // c.f0))
    B = c.buffer_len
    budget = min(8.0, 200.0 / max(1, args.steps + args.warmup))
    strain = strain[:, :hist_s * c.f0 + (args.steps + args.warmup) * B]
    value, s_per_step, sample = time_oracle(banks, strain, B, c.f0, budget, args.steps, args.warmup, len(plan))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * s_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(cfg_no, c, plan, bool(args.banks) and args.banks < c.n_banks),
            "run": {"history_s": hist_s, "note": "each step = one buffer of a bounded sample of the workload's chirp-SVD banks"},
            "cpu_baseline": cpu_baseline_record(value, sample),
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------------
# the CUDA arm
# ---------------------------------------------------------------------------------------------------------
def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured (MEASURED_PEAKS.json)"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "sm_max_mhz": 1965.0}, "fallback (B200_PROFILING.md)"


def ncu_traffic(cfg_no, precision, stage):
    """dram bytes per launch of a stage's kernel from the committed ncu captures (profiles/ncu_traffic.json), keyed by
    (config, precision, stage); None when no capture of that config exists -- never another config's number."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.json")) as f:
            return json.load(f).get(f"config{cfg_no}", {}).get(precision, {}).get(stage)
    except (OSError, ValueError):
        return None


def roofline_record(cfg_no, precision, per_stage, work):
    peaks, peak_src = measured_peaks()
    dom = max(per_stage, key=per_stage.get)
    dom_s = per_stage[dom] / 1e3
    ffma = precision == "ffma"
    # algorithmic work of the dominant kernel per launch: flop in the paper's order
    algo = {"a2_correlate": work[2], "a3_reconstruct_a5_peaks": work[3], "a4_upsample_basis": work[4]}
    executed = {"a2_correlate": work[0], "a3_reconstruct_a5_peaks": work[1]}
    if dom in ("a2_correlate", "a3_reconstruct_a5_peaks"):
        if ffma:
            # dense contraction executed on the FP32 CUDA cores: peak = 148 SM x 128 FFMA lanes x 2 flop x max SM clock
            peak = 148 * 128 * 2 * peaks.get("sm_max_mhz", 1965.0) * 1e6 / 1e12
            bound, peak_note = "alu", "148 SM x 128 lanes x 2 x sm_max_mhz (derived, DESIGN.md)"
        else:
            # fp16 and bf16 share one tcgen05 kind::f16 rate: nominal ratio 1.0 to the measured bf16 peak (sustained:
            # the kernel is timed inside a long step)
            peak = float(peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"]))
            bound, peak_note = "tensor", f"bf16_tflops_sustained x 1.0 (fp16 = bf16 rate), {peak_src}"
        roof = {"bound": bound, "kernel": dom, "achieved": algo[dom] / dom_s / 1e12, "peak": peak, "unit": "TFLOP/s",
                "frac": algo[dom] / dom_s / 1e12 / peak, "traffic": None,
                "executed_tflops": executed[dom] / dom_s / 1e12, "executed_frac": executed[dom] / dom_s / 1e12 / peak,
                "peak_source": peak_note}
    else:
        byt = work[6] if dom == "a4_upsample_basis" else 0.0
        peak = float(peaks["hbm_gbs"])
        roof = {"bound": "hbm", "kernel": dom, "achieved": byt / dom_s / 1e9, "peak": peak, "unit": "GB/s",
                "frac": byt / dom_s / 1e9 / peak, "traffic": None, "peak_source": peak_src}
    roof["traffic"] = ncu_traffic(cfg_no, precision, dom)
    if roof["traffic"] is None:
        roof["traffic_note"] = "no ncu --set full capture of this config/kernel at this commit (profiles/ncu_traffic.json)"
    roof["ms_per_launch"] = per_stage[dom]
    roof["stage_ms_per_push"] = per_stage
    roof["stage_share"] = {k: v / max(sum(per_stage.values()), 1e-12) for k, v in per_stage.items()}
    # every tensor/HBM stage against its own roofline (the dominant one is repeated above)
    tpeak = float(peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"]))
    roof["per_stage"] = {}
    for k in ("a2_correlate", "a3_reconstruct_a5_peaks"):
        if per_stage.get(k, 0) > 0 and not ffma:
            roof["per_stage"][k] = {"algorithmic_tflops": algo[k] / per_stage[k] / 1e9, "frac": algo[k] / per_stage[k] / 1e9 / tpeak,
                                    "executed_frac": executed[k] / per_stage[k] / 1e9 / tpeak}
    if per_stage.get("a4_upsample_basis", 0) > 0:
        roof["per_stage"]["a4_upsample_basis"] = {"gbs_on_intermediate_bytes": work[6] / per_stage["a4_upsample_basis"] / 1e6,
                                                  "frac_of_hbm": work[6] / per_stage["a4_upsample_basis"] / 1e6 / float(peaks["hbm_gbs"])}
    return roof


def measure_config(lib, torch, dist, dev, local_rank, rank, world, cfg_no, K, W, precision, banks_limit, no_flush,
                   shared=None, keep_real=False):
    """Build the stream of one config and time it.  Returns (record, kept) where kept = dict(handles, Ms, real banks) so
    a config with the same banks (config 4 = config 3 at another buffer length) can reuse the uploaded banks."""
    from workloads import make_strain, random_bank
    c, plan = bank_plan(cfg_no, banks_limit)
    B, f0 = c.buffer_len, c.f0
    info = {}
    t_build0 = time.perf_counter()
    if shared is not None:
        st = lib.LloidStream(None, c.n_det, B, precision=PREC[precision], device=f"cuda:{local_rank}",
                             bank_handles=shared["handles"], Ms=shared["Ms"])
        descr, keep = shared["descr"], shared["real"]
    else:
        descr, keep = [], []

        def gen():
            for bank in iter_banks(cfg_no, plan, descr, info):
                if descr[-1].startswith("real") and keep_real:
                    keep.append(bank)
                yield bank
        st = lib.LloidStream(gen(), c.n_det, B, precision=PREC[precision], device=f"cuda:{local_rank}")
    build_s = time.perf_counter() - t_build0
    n_total = 4 * K + W                        # device-timed K, end-to-end K (synchronous and pipelined), stage-timed K
    n_seconds = -(-n_total * B // f0)
    strain = np.stack([make_strain(c.seed(det) + 100 * rank, n_seconds * f0) for det in range(c.n_det)])[:, :n_total * B]
    units_per_step = st.Mtot * c.n_det * (B / f0)
    pool = torch.from_numpy(strain.reshape(c.n_det, n_total, B).transpose(1, 0, 2).copy()).to(dev)   # [step][det][B]
    work = st.work_per_push()
    # L2 policy: the operands (U, R) and intermediates one push touches either exceed the 126 MB L2 several times
    # over (configs 3-5) or the L2 is flushed between steps by writing 256 MiB (configs 1-2)
    touched = work[5] + work[6] / 2
    do_flush = (not no_flush) and touched < 4 * 126e6
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device=dev) if do_flush else None
    l2_note = ("flushed between steps (256 MiB memset, untimed)" if do_flush else
               ("warm (--no-flush)" if no_flush and touched < 4 * 126e6 else
                f"not flushed: one push touches {touched / 1e6:.0f} MB of operands/intermediates (> 4x the 126 MB L2)"))

    def flush():
        if do_flush:
            flush_buf.zero_()

    step = 0
    for _ in range(W):
        flush(); st.push_device(pool[step]); step += 1
    torch.cuda.synchronize()
    sampler = ClockSampler(local_rank)
    sampler.start()
    ev0 = [torch.cuda.Event(enable_timing=True) for _ in range(K)]
    ev1 = [torch.cuda.Event(enable_timing=True) for _ in range(K)]
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    wall0 = time.perf_counter()
    host_ms = []
    for i in range(K):                                                        # ---- device-timed region
        flush()
        ev0[i].record()
        h0 = time.perf_counter()
        st.push_device(pool[step]); step += 1
        host_ms.append(1e3 * (time.perf_counter() - h0))
        ev1[i].record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    wall = time.perf_counter() - wall0
    clocks = sampler.stop()
    ms = [a.elapsed_time(b) for a, b in zip(ev0, ev1)]
    t_dev = max_over_ranks(sum(ms) / 1e3, dev, world)

    # ---- per-stage device times (CUDA events recorded by the library on its stream) for the roofline: K more steps right
    #      after the timed ones (later in the run the board approaches its power cap and the stages would read slower)
    st.set_stage_timing(True)
    for i in range(K):
        flush(); st.push_device(pool[step]); step += 1
    n_cov, stage_ms = st.stage_times()
    st.set_stage_timing(False)

    # ---- end to end through the C ABI with HOST buffers (pinned): H2D strain + push + D2H peaks per step
    t_e2e = 0.0
    for i in range(K):
        st.strain_host.copy_(pool[step].cpu()); step += 1                     # untimed: stage the next buffer in pinned memory
        flush()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        st.push_host()
        t_e2e += time.perf_counter() - t0
    t_e2e = max_over_ranks(t_e2e, dev, world)
    # the same, pipelined (lloid_stream_push_host_async: the peaks of push n travel to the host while push n + 1 computes).
    # Only where no L2 flush between steps is needed (the flush needs a device synchronisation per step).
    t_pipe = None
    if not do_flush:
        xs = [pool[step + i].cpu().pin_memory() for i in range(K)]
        outs = [torch.zeros_like(st.peaks_host).pin_memory() for _ in range(2)]
        step += K
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for i in range(K):
            st.push_host_async(xs[i], outs[i & 1])
        st.host_sync()
        t_pipe = max_over_ranks(time.perf_counter() - t0, dev, world)

    # ---- "empty push": the same launch sequence on a one-template, 64-tap bank = launch overhead per push
    tiny = lib.LloidStream([random_bank(1, 1, [(f0, 64, 1)], f0=f0).as_f32()], c.n_det, B, precision=PREC[precision],
                           device=f"cuda:{local_rank}")
    e0 = [torch.cuda.Event(enable_timing=True) for _ in range(40)]
    e1 = [torch.cuda.Event(enable_timing=True) for _ in range(40)]
    for i in range(40):
        e0[i].record(); tiny.push_device(pool[i % n_total]); e1[i].record()
    torch.cuda.synchronize()
    empty_ms = float(np.median([a.elapsed_time(b) for a, b in zip(e0[8:], e1[8:])]))
    tiny.close()

    # ---- event identification on the peaks of the last push (coincidence + clustering): not part of the
    #      timed step, reported beside it
    ev_ms = None
    if c.n_det >= 2:
        dt = np.full((c.n_det, c.n_det), int(math.ceil(0.0323 * f0)), dtype=np.int32)
        np.fill_diagonal(dt, 0)
        st.events(dt)
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g0.record()
        for _ in range(5):
            lib.binding.lloid_stream_events(st.handle, st.peaks_dev.data_ptr(), dt, st.events_dev.data_ptr())
        g1.record(); torch.cuda.synchronize()
        ev_ms = g0.elapsed_time(g1) / 5

    launches = st.launches_per_push
    d2h = int(st.peaks_host.numel() * st.peaks_host.element_size())
    handles, Ms = st.release_banks() if shared is None else (None, None)      # the caller owns (and frees) the bank handles
    st.close()
    del pool, flush_buf
    torch.cuda.empty_cache()

    per_stage = {k: v / max(n_cov, 1) for k, v in stage_ms.items()}            # ms per push
    rec = {
        "metric": METRIC, "value": whole_job_value(world, units_per_step, K, t_dev), "unit": UNIT, "n_gpus": world,
        "steps": K, "warmup": W, "ms_per_step": 1e3 * t_dev / K, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": PREC_DTYPE[precision], "data": "synthetic",
        "config": config_dict(cfg_no, c, plan, bool(banks_limit) and banks_limit < c.n_banks),
        "run": {"slices": descr[:2] + descr[-2:], "precision": precision, "l2": l2_note,
                "timing": "sum of per-step CUDA-event intervals (push only), max over ranks",
                "multi_gpu": "independent replicas of the workload, no data-path collective",
                "stream_build_s": build_s, "banks_shared_with": (shared or {}).get("cfg"), **info},
        "e2e": {"value": whole_job_value(world, units_per_step, K, t_pipe if t_pipe is not None else t_e2e), "unit": UNIT,
                "h2d_bytes_per_step": c.n_det * B * 4, "d2h_bytes_per_step": d2h,
                "ms_per_step": 1e3 * (t_pipe if t_pipe is not None else t_e2e) / K,
                "mode": ("pipelined: K x lloid_stream_push_host_async + lloid_stream_host_sync, pinned host buffers, two pushes in "
                         "flight (every step's H2D strain copy and D2H peaks copy inside the timed region)" if t_pipe is not None else
                         "synchronous: lloid_stream_push_host per step (L2 flushed between steps)"),
                "synchronous_value": whole_job_value(world, units_per_step, K, t_e2e), "synchronous_ms_per_step": 1e3 * t_e2e / K},
        "gpu_launches": launches * K, "wall_ms_timed_region": 1e3 * wall,
        "ms_step_min_med_max": [min(ms), float(np.median(ms)), max(ms)],
        "latency_ms": {"device_p50": float(np.percentile(ms, 50)), "device_p99": float(np.percentile(ms, 99)),
                       "device_max": max(ms), "host_launch_p50": float(np.percentile(host_ms, 50)),
                       "host_launch_p99": float(np.percentile(host_ms, 99)), "empty_push_device_p50": empty_ms,
                       "realtime_budget_ms": 1e3 * B / f0,
                       "note": "per-push device time (CUDA events around one lloid_stream_push), host time of the call, and the "
                               "device time of a push on a one-template 64-tap bank (launch overhead of the kernel sequence)"},
        "clocks": clocks, "roofline": roofline_record(cfg_no, precision, per_stage, work),
        "events_stage_ms": ev_ms,
    }
    kept = {"cfg": cfg_no, "handles": handles, "Ms": Ms, "descr": descr, "real": keep}
    return rec, kept


def free_kept(lib, kept):
    for h in (kept or {}).get("handles") or []:
        lib.lloid_bank_destroy(h)


def run_plumbing_check(args):
    """CPU-only: launcher -> ranks -> gloo process group -> barrier -> max over ranks -> one rank-0 line (no filtering)."""
    import torch
    import torch.distributed as dist
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:
        dist.init_process_group("gloo")
        dist.barrier()
    t = max_over_ranks(0.010 * (rank + 1), torch.device("cpu"), world)       # the last rank is the slow one
    if rank == 0:
        print(json.dumps({"plumbing_check": True, "n_gpus": world, "gpus_arg": args.gpus, "t": t,
                          "value": whole_job_value(world, 64.0, args.steps, t), "scaling": "weak"}), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_ours(args):
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the LLOID path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    import paper_2511_04730_b200 as lib

    K, W = args.steps, args.warmup
    head_cfg = args.config or HEADLINE_CONFIG
    want_oracle = not args.no_cpu_baseline and world == 1
    line, kept = measure_config(lib, torch, dist, dev, local_rank, rank, world, head_cfg, K, W, args.precision, args.banks,
                                args.no_flush, keep_real=want_oracle)
    real_head = kept["real"]
    free_kept(lib, kept)
    if not args.config and not args.no_nested:
        others, kept3 = {}, None
        for cfg_no in NESTED_CONFIGS:
            k_cfg = max(K, 200) if cfg_no == 4 else K                         # p99 of the 1/16 s pushes needs >= 200 samples
            shared = kept3 if cfg_no == 4 and kept3 and kept3.get("handles") else None
            rec, kept_n = measure_config(lib, torch, dist, dev, local_rank, rank, world, cfg_no, k_cfg, W, args.precision, 0,
                                         args.no_flush, shared=shared, keep_real=(cfg_no == 3))
            others[f"config{cfg_no}"] = rec
            if cfg_no == 3:
                kept3 = kept_n
            elif shared is None:
                free_kept(lib, kept_n)
        free_kept(lib, kept3)
        line["other_configs"] = others
    if rank == 0:
        if want_oracle and real_head:
            from workloads import CONFIGS, make_strain
            c = CONFIGS[head_cfg]
            hist_s, n_buf = 4, 5
            n = hist_s * c.f0 + n_buf * c.buffer_len
            strain_o = np.stack([make_strain(c.seed(det), -(-n // c.f0) * c.f0) for det in range(c.n_det)])[:, :n]
            v, _, sample = time_oracle(real_head, strain_o, c.buffer_len, c.f0, 4.0, n_buf, 0, line["config"]["n_banks"])
            line["cpu_baseline"] = cpu_baseline_record(v, sample)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    env_world = os.environ.get("WORLD_SIZE")
    if args.gpus > 1 and env_world is None:
        # not yet under a launcher: start one rank per GPU (the driver's own torchrun command lands in the branch below)
        cmd = launcher_command(args.gpus, sys.argv[1:])
        os.execv(cmd[0], cmd)
    if env_world is not None and int(env_world) != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but the launcher started WORLD_SIZE={env_world} ranks; "
                         f"run `python bench.py --gpus N` (it launches torch.distributed.run itself) or give both the same N")
    if args.plumbing_check:
        run_plumbing_check(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
