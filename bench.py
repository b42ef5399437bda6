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
    ap.add_argument("--precision", default=os.environ.get("LLOID_BENCH_PRECISION", "split"), choices=list(PREC))
    ap.add_argument("--banks", type=int, default=0, help="debug: use only the first n banks (0 = all; marks the run as reduced)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-flush", action="store_true", help="keep L2 warm between steps (reported in config)")
    return ap.parse_args()


# ---------------------------------------------------------------------------------------------------------
# workload
# ---------------------------------------------------------------------------------------------------------
N_REAL_BANKS = 4        # configs with many banks: this many real chirp-SVD banks, the rest shape-faithful stand-ins


def _real_bank(args):
    """One chirp-SVD bank of the config.  Generation is deterministic and slow for 1000-template banks (0.5-2 min),
    so the result is memoised under /tmp (an input cache only: a miss just recomputes the same arrays)."""
    cfg_no, b = args
    import pickle
    from workloads import CONFIGS
    c = CONFIGS[cfg_no]
    path = os.path.join("/tmp", "lloid_bank_cache", f"seed{c.seed(999)}_M{c.M}_nb{c.n_banks}_T{int(c.T_max)}_b{b}.pkl")
    try:
        with open(path, "rb") as f:
            return b, pickle.load(f)
    except Exception:
        pass
    bank = c.bank(b, method="gram" if c.M >= 1000 else "svd").as_f32()
    try:
        os.makedirs(os.path.dirname(path), exist_ok=True)
        with open(path + f".{os.getpid()}", "wb") as f:
            pickle.dump(bank, f, protocol=4)
        os.replace(path + f".{os.getpid()}", path)
    except Exception:
        pass
    return b, bank


def bank_plan(cfg_no, n_banks_limit):
    """(config, list of bank descriptions).  Configs 1-2: every bank is the config's chirp-SVD bank.  Configs 3-5
    (100-1000 banks; one SVD bank takes 0.5-1 min of host time): N_REAL_BANKS evenly spaced real banks; every other
    bank keeps its REAL slice layout (rates, taps, delays from its own chirp masses) and takes the basis counts L^s of
    the nearest real bank, with seeded random orthonormal U and random R (SURVEY.md section 8d "scale handling")."""
    from workloads import CONFIGS
    c = CONFIGS[cfg_no]
    nb = c.n_banks if not n_banks_limit else min(n_banks_limit, c.n_banks)
    if nb <= 8:
        return c, [("real", b) for b in range(nb)]
    real = sorted(set(int(round(i * (nb - 1) / (N_REAL_BANKS - 1))) for i in range(N_REAL_BANKS)))
    return c, [("real", b) if b in real else ("standin", b, min(real, key=lambda r: abs(r - b))) for b in range(nb)]


def iter_banks(cfg_no, plan, describe=None):
    """Yield the planned banks one at a time (the caller uploads each and drops it)."""
    import multiprocessing as mp
    from workloads import CONFIGS, random_bank
    c = CONFIGS[cfg_no]
    mcs = c.mchirps()
    real_ids = [p[1] for p in plan if p[0] == "real"]
    if len(real_ids) > 1 and c.M >= 1000:
        with mp.get_context("fork").Pool(min(len(real_ids), os.cpu_count() or 1)) as pool:
            real = dict(pool.map(_real_bank, [(cfg_no, b) for b in real_ids]))
    else:
        real = dict(_real_bank((cfg_no, b)) for b in real_ids)
    for p in plan:
        if p[0] == "real":
            bank = real[p[1]]
        else:
            _, b, src = p
            T, lay = c.layout(b, mcs)
            Ls = [s.n_basis for s in real[src].slices]
            shape = [(rate, (e - s0) // (c.f0 // rate), Ls[min(i, len(Ls) - 1)]) for i, (rate, s0, e) in enumerate(lay)]
            bank = random_bank(c.seed(b), c.M, shape, f0=c.f0).as_f32()
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
    from workloads import make_strain
    c, plan = bank_plan(args.config, args.banks)
    B, f0 = c.buffer_len, c.f0
    descr = []
    keep = []                                  # banks kept on the host only when the oracle baseline needs them
    def gen():
        for bank in iter_banks(args.config, plan, descr):
            if descr[-1].startswith("real"):
                keep.append(bank)
            yield bank
    st = lib.LloidStream(gen(), c.n_det, B, precision=PREC[args.precision], device=f"cuda:{local_rank}")
    banks = keep
    n_seconds = -(-n_total * B // f0)
    strain = np.stack([make_strain(c.seed(det) + 100 * rank, n_seconds * f0) for det in range(c.n_det)])[:, :n_total * B]
    units_per_step = st.Mtot * c.n_det * (B / f0)
    pool = torch.from_numpy(strain.reshape(c.n_det, n_total, B).transpose(1, 0, 2).copy()).to(dev)   # [step][det][B]
    work = st.work_per_push()
    # L2 policy: the operands (U, R) and intermediates one push touches either exceed the 126 MB L2 several times
    # over (configs 3-5) or the L2 is flushed between steps by writing 256 MiB (configs 1-2)
    touched = work[5] + work[6] / 2
    do_flush = (not args.no_flush) and touched < 4 * 126e6
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device=dev) if do_flush else None
    l2_note = ("flushed between steps (256 MiB memset, untimed)" if do_flush else
               ("warm (--no-flush)" if args.no_flush and touched < 4 * 126e6 else
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

    # ---- "empty push": the same five-kernel launch sequence on a one-template, 64-tap bank = launch overhead per push
    from workloads import random_bank
    tiny = lib.LloidStream([random_bank(1, 1, [(f0, 64, 1)], f0=f0).as_f32()], c.n_det, B, precision=PREC[args.precision],
                           device=f"cuda:{local_rank}")
    e0 = [torch.cuda.Event(enable_timing=True) for _ in range(40)]
    e1 = [torch.cuda.Event(enable_timing=True) for _ in range(40)]
    for i in range(40):
        e0[i].record(); tiny.push_device(pool[i % n_total]); e1[i].record()
    torch.cuda.synchronize()
    empty_ms = float(np.median([a.elapsed_time(b) for a, b in zip(e0[8:], e1[8:])]))
    tiny.close()

    # ---- per-stage device times (CUDA events recorded by the library on its stream) for the roofline
    st.set_stage_timing(True)
    for i in range(K):
        flush(); st.push_device(pool[step]); step += 1
    n_cov, stage_ms = st.stage_times()
    st.set_stage_timing(False)
    launches = st.launches_per_push
    st.close()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    line = assemble(args, c, descr, world, K, W, units_per_step, t_dev, ms, wall, t_e2e, stage_ms, n_cov, work, launches, clocks,
                    l2_note, host_ms, empty_ms)
    if not args.no_cpu_baseline and world == 1 and banks:
        hist_s = 4
        strain_o = np.stack([make_strain(c.seed(det), (hist_s + 1) * f0) for det in range(c.n_det)])[:, :hist_s * f0 + B]
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


def assemble(args, c, descr, world, K, W, units_per_step, t_dev, ms, wall, t_e2e, stage_ms, n_cov, work, launches, clocks,
             l2_note, host_ms, empty_ms):
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
    banks = descr
    return {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": 1e3 * t_dev / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": PREC_DTYPE[args.precision], "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[{args.config - 1}] ({c.name})" + (" REDUCED (--banks)" if reduced else ""),
                   "n_banks": len(descr), "templates_per_bank": c.M, "n_detectors": c.n_det, "buffer_len": c.buffer_len,
                   "banks": (f"{sum(d.startswith('real') for d in descr)} chirp-SVD banks + "
                             f"{sum(d.startswith('standin') for d in descr)} shape-faithful stand-ins (real slice layout, L^s of the "
                             "nearest SVD bank, random orthonormal U / random R)"),
                   "slices": descr[:2] + descr[-2:], "precision": args.precision, "l2": l2_note,
                   "timing": "sum of per-step CUDA-event intervals (push only), max over ranks",
                   "multi_gpu": "independent replicas of the workload, no data-path collective"},
        "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": c.n_det * c.buffer_len * 4,
                "d2h_bytes_per_step": int(c.n_det * len(descr) * c.M * 12), "ms_per_step": 1e3 * t_e2e / K},
        "gpu_launches": launches * K, "wall_ms_timed_region": 1e3 * wall, "ms_step_min_med_max": [min(ms), float(np.median(ms)), max(ms)],
        "latency_ms": {"device_p50": float(np.percentile(ms, 50)), "device_p99": float(np.percentile(ms, 99)),
                       "device_max": max(ms), "host_launch_p50": float(np.percentile(host_ms, 50)),
                       "host_launch_p99": float(np.percentile(host_ms, 99)), "empty_push_device_p50": empty_ms,
                       "note": "per-push device time (CUDA events around one lloid_stream_push), host time of the call, and the device time of a push on a one-template 64-tap bank (launch overhead of the five-kernel sequence)"},
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
