"""CPU-side tests of the boundary: liblloid.so loads, exports every symbol include/lloid.h declares, validates its
arguments before touching the device (no compute calls here), and the multi-rank bench plumbing works over gloo."""
import ctypes as C
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    sys.path.insert(0, ROOT)
    from paper_2511_04730_b200 import build
    build.build()
    import paper_2511_04730_b200 as lib
    return lib


def declared_functions():
    src = open(os.path.join(ROOT, "include", "lloid.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lloid_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_are_exported_and_bound(lib):
    names = declared_functions()
    assert "lloid_bank_create" in names and "lloid_stream_push" in names and "lloid_state_reset" in names
    so = C.CDLL(lib.LIB_PATH)
    for n in names:
        assert hasattr(so, n), f"{n} declared in include/lloid.h but not exported by liblloid.so"
        assert n in lib.EXPORTS, f"{n} has no binding in paper_2511_04730_b200/binding.py"
    assert lib.lloid_version().startswith("lloid-b200")


def test_library_is_sm100a_with_tcgen05_and_tma(lib):
    """The product path is hand-written sm_100a code: the SASS must contain tcgen05 MMA, TMEM loads and TMA."""
    out = subprocess.run(["cuobjdump", "-sass", lib.LIB_PATH], capture_output=True, text=True)
    if out.returncode != 0:
        pytest.skip("cuobjdump unavailable")
    assert "sm_100a" in out.stdout
    for mnemonic in ("UTCHMMA", "LDTM", "UTMALDG"):
        assert mnemonic in out.stdout, mnemonic


def _slice(rate, n_taps, L, delay, M, ok_arrays=True):
    U = np.zeros((L, n_taps), np.float32)
    R = np.zeros((2 * M, L), np.float32)
    return dict(rate_hz=rate, n_taps=n_taps, n_basis=L, delay=delay, basis=U, recon=R)


def test_bank_create_rejects_bad_slice_tables(lib):
    M = 4
    bad = {
        "rate not f0/2^k": [_slice(2048, 64, 2, 0, M), _slice(1000, 64, 2, 32, M)],
        "delay[0] != 0": [_slice(2048, 64, 2, 5, M)],
        "slice 0 not at f0": [_slice(1024, 64, 2, 0, M)],
        "rates increase": [_slice(2048, 64, 2, 0, M), _slice(1024, 64, 2, 32, M), _slice(2048, 64, 2, 160, M)],
        "slices do not abut": [_slice(2048, 64, 2, 0, M), _slice(1024, 64, 2, 40, M)],
    }
    for why, sl in bad.items():
        with pytest.raises(lib.LloidError) as e:
            lib.lloid_bank_create(2048, M, sl, precision=lib.LLOID_PREC_FP32_FFMA)
        assert e.value.code == lib.LLOID_EINVAL, why
        assert lib.lloid_last_error() != ""
    with pytest.raises(lib.LloidError) as e:       # f0 not a power of two
        lib.lloid_bank_create(3000, M, [_slice(3000, 64, 2, 0, M)])
    assert e.value.code == lib.LLOID_EINVAL
    with pytest.raises(lib.LloidError) as e:       # unknown precision
        lib.lloid_bank_create(2048, M, [_slice(2048, 64, 2, 0, M)], precision=7)
    assert e.value.code == lib.LLOID_EINVAL


def test_bank_create_enforces_the_causality_condition(lib):
    """a down-sampled slice must be delayed by at least its decimator + upsample-chain look-ahead:
    delay_s >= n_down + H (H = 9 samples for one x2 stage).  64 f0 taps -> delay 32 at 1024 Hz < 32 + 9."""
    M = 4
    with pytest.raises(lib.LloidError) as e:
        lib.lloid_bank_create(2048, M, [_slice(2048, 64, 2, 0, M), _slice(1024, 64, 2, 32, M)],
                              precision=lib.LLOID_PREC_FP32_FFMA)
    assert e.value.code == lib.LLOID_ELATENCY
    assert "delay" in lib.lloid_last_error()


def test_null_and_state_errors_without_a_device(lib):
    assert lib.binding._lib.lloid_stream_push(None, None, None, None, 0) == lib.LLOID_EINVAL
    assert lib.binding._lib.lloid_state_reset(None) == lib.LLOID_EINVAL
    assert lib.binding._lib.lloid_stream_samples_pushed(None) == -1
    out = C.c_void_p()
    assert lib.binding._lib.lloid_stream_create(C.byref(out), None, 0, 1, 2048, None) == lib.LLOID_EINVAL
    o = lib.lloid_options_default()
    assert (o.n_down, o.n_up, o.precision) == (32, 8, lib.LLOID_PREC_F16_SPLIT)
    assert o.trigger_overlap == 0 and o.threshold == 0.0
    # the calls around the path validate their arguments before touching a device
    L = lib.binding._lib
    assert L.lloid_stream_events(None, None, None, None) == lib.LLOID_EINVAL
    assert L.lloid_stream_push_host_async(None, None, None) == lib.LLOID_EINVAL and L.lloid_stream_host_sync(None) == lib.LLOID_EINVAL
    assert L.lloid_stream_xi2(None, None) == lib.LLOID_EINVAL
    assert L.lloid_bank_set_autocorrelation(None, None, 175) == lib.LLOID_EINVAL
    assert L.lloid_xi2_series(None, 1, 1, None, None, 175, None, None) == lib.LLOID_EINVAL
    assert L.lloid_whitener_push(None, None, None, None) == lib.LLOID_EINVAL
    w = C.c_void_p()
    for bad in ((1, 16384, 2000, 65536, 16384, 7, 64), (1, 16384, 2048, 65536, 16384, 6, 64), (1, 16384, 2048, 65535, 16384, 7, 64),
                (0, 16384, 2048, 65536, 16384, 7, 64), (1, 16384, 2048, 65536, 40000, 7, 64)):
        assert L.lloid_whitener_create(C.byref(w), *bad, None) == lib.LLOID_EINVAL and "whitener_create" in lib.lloid_last_error()
    n = C.c_int32()
    assert L.lloid_svd_slice(None, 4, 4, 0.9999, 4, C.byref(n), None, None, None, None, None) == lib.LLOID_EINVAL
    assert L.lloid_svd_slice_noalloc(None, 4, 4, 0.9999, 4, C.byref(n), None, None, None, None, None) == lib.LLOID_EINVAL
    assert L.lloid_whitener_hop_in(None) == -1


def test_product_path_never_imports_the_oracle():
    """The oracle is test infrastructure: nothing under the package (or the input generators) may import it."""
    for top in ("paper_2511_04730_b200", "workloads"):
        for dirpath, _, files in os.walk(os.path.join(ROOT, top)):
            for f in files:
                if f.endswith((".py", ".cu", ".cuh", ".h")):
                    txt = open(os.path.join(dirpath, f)).read()
                    assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), os.path.join(dirpath, f)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            assert "paper_2511_04730_b200" not in re.sub(r'""".*?"""', "", open(os.path.join(ROOT, "oracle", f)).read(), flags=re.S)


_GLOO_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
t_local = 0.010 * (rank + 1)                       # rank 1 is the slow one
t = bench.max_over_ranks(t_local, torch.device("cpu"), world)
c, banks, strain = bench.build_workload(1, 0, 1, rank)
val = bench.whole_job_value(world, 64 * 1 * 1.0, 5, t)
if rank == 0:
    print(json.dumps({{"t": t, "value": val, "seed0": float(strain[0, 0])}}))
else:
    print(json.dumps({{"seed1": float(strain[0, 0])}}), file=sys.stderr)
dist.destroy_process_group()
"""


def test_multi_rank_bench_plumbing_gloo(tmp_path):
    """world_size 2 over gloo: the timed value is the max over ranks, the throughput is the whole-job aggregate of
    independent replicas, and every rank draws its own strain (no data-path collective exists to test)."""
    import json
    script = tmp_path / "worker.py"
    script.write_text(_GLOO_WORKER.format(root=ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29577")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                        "--master-addr", "127.0.0.1", "--master-port", "29577", str(script)],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    line = [ln for ln in r.stdout.splitlines() if ln.startswith("{")][-1]
    res = json.loads(line)
    assert abs(res["t"] - 0.020) < 1e-9                       # max over ranks
    assert abs(res["value"] - 2 * 64 * 5 / 0.020) < 1e-6      # whole-job aggregate
    seed1 = [json.loads(ln) for ln in r.stderr.splitlines() if ln.startswith('{"seed1"')]
    assert seed1 and seed1[-1]["seed1"] != res["seed0"]       # replicas filter different strain


def test_bench_gpus_flag_launches_ranks_itself():
    """`python bench.py --gpus 2` (no torchrun around it) must start 2 ranks on its own: the plumbing check runs the
    launcher -> rank environment -> process group (gloo) -> barrier -> max over ranks -> one rank-0 line path without
    any filtering, and the printed n_gpus is the number of ranks the process group saw."""
    import json
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    env["MASTER_PORT"] = "29591"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "5", "--plumbing-check"],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                     # rank 0 alone prints
    res = json.loads(lines[0])
    assert res["n_gpus"] == 2 and res["gpus_arg"] == 2
    assert abs(res["t"] - 0.020) < 1e-9                        # max over ranks
    assert abs(res["value"] - 2 * 64 * 5 / 0.020) < 1e-6       # whole-job aggregate of 2 replicas


def test_bench_refuses_a_rank_count_that_contradicts_gpus():
    """Under a launcher whose WORLD_SIZE differs from --gpus the bench exits non-zero instead of printing a wrong n_gpus."""
    env = dict(os.environ, WORLD_SIZE="2", RANK="0", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "1", "--plumbing-check"],
                       capture_output=True, text=True, env=env, timeout=120)
    assert r.returncode != 0 and "--gpus" in r.stderr


def test_bench_plan_is_deterministic_and_names_the_headline():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.HEADLINE_CONFIG == 5 and bench.parse([]).config == 0
    c, plan = bench.bank_plan(5)
    assert len(plan) == 1000 and bench.config_dict(5, c, plan)["workload"].startswith("BASELINE.json configs[4]")
    real = [p[1] for p in plan if p[0] == "real"]
    assert {0, 333, 666, 999} <= set(real) and 4 < len(real) <= 8
    inj_banks = [i.bank for i in c.injections(bench.parity_seconds(c))]
    assert set(real) - {0, 333, 666, 999} <= set(inj_banks)                     # the extra real banks are injected banks
    assert plan == bench.bank_plan(5)[1]
    for p in plan:
        assert p[0] == "real" or p[2] in real
