#!/usr/bin/env python
"""bench.py -- LLOID hot-path throughput on B200 (driver contract).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2] [--precision split]

A STEP is one lloid_stream_push of one buffer (config 2: 1 s = 2048 samples) of every detector against every
bank: a1 decimate -> a2 basis correlation -> a4 upsample -> a3 reconstruction -> a5 peaks.  The metric is
BASELINE.json's: template*detector*data-seconds filtered per wall-second.  Workload = BASELINE.json configs[1]
(4 SVD banks x 500 chirp templates, 2 detectors, 1 s buffers), seeded synthetic inputs from workloads/.
Prints ONE JSON line on rank 0.  `--impl reference` times the float64 CPU oracle (oracle/) on the host cores.
"""
import argparse
import json
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
PREC_DTYPE = {"ffma": "f32", "f16": "f16 operands, f32 accumulate", "split": "f16 hi+lo split operands (3 MMAs), f32 accumulate"}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config number (1-based); default 2 = configs[1]")
    ap.add_argument("--precision", default=os.environ.get("LLOID_BENCH_PRECISION", "ffma"), choices=list(PREC))
    ap.add_argument("--banks", type=int, default=0, help="debug: use only the first n banks (0 = all; marks the run as reduced)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-flush", action="store_true", help="keep L2 warm between steps (reported in config)")
    return ap.parse_args()


# ---------------------------------------------------------------------------------------------------------
# workload
# ---------------------------------------------------------------------------------------------------------
def build_workload(cfg_no, n_banks_limit, seconds, rank=0):
    """Banks (float32-rounded SVD banks of the config) and [n_det][seconds*f0] strain, seeded (DESIGN.md recipe)."""
    from workloads import CONFIGS, make_strain
    c = CONFIGS[cfg_no]
    mcs = c.mchirps()
    nb = c.n_banks if not n_banks_limit else min(n_banks_limit, c.n_banks)
    banks = [c.bank(b, method="gram" if c.M >= 1000 else "svd", mcs=mcs).as_f32() for b in range(nb)]
    # white N(0,1) strain per detector; ranks > 0 (weak scaling replicas) shift the detector seeds
    strain = np.stack([make_strain(c.seed(det) + 100 * rank, seconds * c.f0) for det in range(c.n_det)])
    return c, banks, strain


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


def time_oracle(banks, strain, B, f0, budget_s, steps=1, warmup=0):
    """Time `steps` oracle steps on a bounded sample: as many leading banks as fit ~budget_s per step."""
    n_det = strain.shape[0]
    hist = strain.shape[1] - (steps + warmup) * B
    assert hist >= 0
    t0 = time.perf_counter()
    oracle_step(banks[:1], strain, hist + B if hist + B <= strain.shape[1] else strain.shape[1], B)   # calibration
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
    return units / dt, dt / steps, f"{nb} of {len(banks)} banks x {n_det} detectors x {steps} buffer(s) of {B} samples, float64 numpy"


def run_reference(args):
    """--impl reference: the oracle as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    hist_s = 4
    c, banks, strain = build_workload(args.config, args.banks, hist_s + args.steps + args.warmup)
    B = c.buffer_len
    budget = min(8.0, 200.0 / max(1, args.steps + args.warmup))
    value, s_per_step, sample = time_oracle(banks, strain, B, c.f0, budget, args.steps, args.warmup)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * s_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"BASELINE.json configs[{args.config - 1}] ({c.name})", "n_banks": len(banks),
                       "templates_per_bank": c.M, "n_detectors": c.n_det, "buffer_len": B, "history_s": hist_s},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": blas_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


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
    n_total = 3 * K + W                        # device-timed K, end-to-end K, stage-timed K
    c, banks, strain = build_workload(args.config, args.banks, n_total, rank)
    B, f0 = c.buffer_len, c.f0
    st = lib.LloidStream(banks, c.n_det, B, precision=PREC[args.precision], device=f"cuda:{local_rank}")
    units_per_step = st.Mtot * c.n_det * (B / f0)
    pool = torch.from_numpy(strain.reshape(c.n_det, n_total, B).transpose(1, 0, 2).copy()).to(dev)   # [step][det][B]
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device=dev)        # 256 MiB > 126 MB L2

    def flush():
        if not args.no_flush:
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
    for i in range(K):                                                        # ---- device-timed region
        flush()
        ev0[i].record()
        st.push_device(pool[step]); step += 1
        ev1[i].record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    wall = time.perf_counter() - wall0
    clocks = sampler.stop()
    ms = [a.elapsed_time(b) for a, b in zip(ev0, ev1)]
    t_dev = max_over_ranks(sum(ms) / 1e3, dev, world)

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

    # ---- per-stage device times (CUDA events recorded by the library on its stream) for the roofline
    st.set_stage_timing(True)
    for i in range(K):
        flush(); st.push_device(pool[step]); step += 1
    n_cov, stage_ms = st.stage_times()
    st.set_stage_timing(False)
    work = st.work_per_push()
    launches = st.launches_per_push
    st.close()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    line = assemble(args, c, banks, world, K, W, units_per_step, t_dev, ms, wall, t_e2e, stage_ms, n_cov, work, launches, clocks)
    if not args.no_cpu_baseline and world == 1:
        hist_s = 4
        _, _, strain_o = build_workload(args.config, args.banks, hist_s + 1)
        v, s_per, sample = time_oracle(banks, strain_o, B, f0, 15.0, 1, 0)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": blas_threads(), "kind": "oracle", "sample": sample}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured (MEASURED_PEAKS.json)"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "sm_max_mhz": 1965.0}, "fallback (B200_PROFILING.md)"


def assemble(args, c, banks, world, K, W, units_per_step, t_dev, ms, wall, t_e2e, stage_ms, n_cov, work, launches, clocks):
    peaks, peak_src = measured_peaks()
    value = whole_job_value(world, units_per_step, K, t_dev)
    e2e = whole_job_value(world, units_per_step, K, t_e2e)
    per_stage = {k: v / max(n_cov, 1) for k, v in stage_ms.items()}            # ms per push
    dom = max(per_stage, key=per_stage.get)
    dom_s = per_stage[dom] / 1e3
    ffma = args.precision == "ffma"
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
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.json")) as f:
            roof["traffic"] = json.load(f).get(args.precision, {}).get(dom)
    except OSError:
        pass
    roof["ms_per_launch"] = per_stage[dom]
    roof["stage_ms_per_push"] = per_stage
    roof["stage_share"] = {k: v / max(sum(per_stage.values()), 1e-12) for k, v in per_stage.items()}
    reduced = bool(args.banks) and args.banks < c.n_banks
    return {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": 1e3 * t_dev / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": PREC_DTYPE[args.precision], "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[{args.config - 1}] ({c.name})" + (" REDUCED (--banks)" if reduced else ""),
                   "n_banks": len(banks), "templates_per_bank": c.M, "n_detectors": c.n_det, "buffer_len": c.buffer_len,
                   "slices": [b.describe() for b in banks[:4]], "precision": args.precision,
                   "l2": "warm (--no-flush)" if args.no_flush else "flushed between steps (256 MiB memset, untimed)",
                   "timing": "sum of per-step CUDA-event intervals (push only), max over ranks",
                   "multi_gpu": "independent replicas of the workload, no data-path collective"},
        "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": c.n_det * c.buffer_len * 4,
                "d2h_bytes_per_step": int(c.n_det * sum(b.M for b in banks) * 12), "ms_per_step": 1e3 * t_e2e / K},
        "gpu_launches": launches * K, "wall_ms_timed_region": 1e3 * wall, "ms_step_min_med_max": [min(ms), float(np.median(ms)), max(ms)],
        "clocks": clocks, "roofline": roof,
    }


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
