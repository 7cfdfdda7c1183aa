"""CPU-side checks of the product: the C-ABI library builds for sm_100a and exports every symbol
include/roadrunner.h declares, fails loudly without a GPU (no CPU fallback), and the host logic
around it (sharding, bench plumbing) is right.  No compute calls here."""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_symbols():
    text = open(os.path.join(ROOT, "include", "roadrunner.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rr_[a-z0-9_]+)\s*\(", text)))


def test_library_builds_and_exports_every_declared_symbol():
    import paper_2009_08500_b200 as rr
    lib = rr.load()
    declared = header_symbols()
    assert len(declared) >= 20
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in roadrunner.h but not exported"
    assert sorted(rr.SYMBOLS) == declared


def test_library_is_sm100a_native():
    import paper_2009_08500_b200 as rr
    rr.load()
    out = subprocess.run(["cuobjdump", "-lelf", rr.library_path()], capture_output=True, text=True)
    if out.returncode != 0:
        pytest.skip("cuobjdump not available")
    assert "sm_100a" in out.stdout


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import paper_2009_08500_b200 as rr
    with pytest.raises(rr.RoadRunnerError) as e:
        rr.rr_create()
    assert e.value.code <= -1000          # a CUDA error, surfaced
    assert "rr_create" in str(e.value)


def test_host_side_argument_checks_need_no_device():
    import paper_2009_08500_b200 as rr
    lib = rr.load()
    assert lib.rr_create(None, None) == -1
    cfg = rr.rr_config(50, 50, 0.7, 1, 50, 0.02, 0.2, 1, 1, 0)       # ng = 1
    h = ctypes.c_void_p()
    assert lib.rr_create(ctypes.byref(cfg), ctypes.byref(h)) == -2
    cfg = rr.rr_config(50, 50, 0.7, 100, 50, 0.2, 0.02, 1, 1, 0)     # k1 < k0
    assert lib.rr_create(ctypes.byref(cfg), ctypes.byref(h)) == -2
    cfg = rr.rr_config(50, 50, 0.7, 100, 50, 0.02, 0.2, 4, 2, 0)     # nkpb not in {1, npb}
    assert lib.rr_create(ctypes.byref(cfg), ctypes.byref(h)) == -2
    assert lib.rr_evaluate(None, None, 7, 1, None, None, None) == -1
    assert lib.rr_num_tiles(None) == -1
    assert rr.error_string(-4).startswith("lc_index")
    assert rr.error_string(0) == "ok"


def test_product_does_not_import_the_oracle():
    """The product path shares no code with the oracle and never imports it."""
    pkg = os.path.join(ROOT, "paper_2009_08500_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "roadrunner_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2009_08500_b200" not in text, f
            assert "from paper_2009_08500_b200" not in text, f


def test_pv_slice_partitions_the_population():
    from paper_2009_08500_b200.shard import pv_slice
    for npv in (0, 1, 7, 16384, 1000003):
        for world in (1, 2, 3, 8):
            edges = [pv_slice(npv, r, world) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == npv
            assert all(a[1] == b[0] for a, b in zip(edges, edges[1:]))
            sizes = [e - b for b, e in edges]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        pv_slice(10, 2, 2)


def _gloo_worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from paper_2009_08500_b200 import shard
    import workloads
    r, w = shard.init_process_group("gloo")
    wl = workloads.make_workload(1, npv=101, npt=50)
    b, e = shard.pv_slice(wl.npv, r, w)
    mine = wl.subset_pv(np.arange(b, e))
    shard.barrier()
    tmax = shard.max_over_ranks(10.0 + r)
    total = shard.sum_over_ranks(float(mine.evaluations))
    q.put((r, b, e, tmax, total, float(mine.pv[:, 0].sum())))
    dist.destroy_process_group()


def test_two_rank_gloo_sharding():
    """world_size 2 on CPU (gloo): ranks own disjoint pv slices, the timing reduce is the max over
    ranks and the unit count the sum - the only communication the path has."""
    import torch.multiprocessing as mp
    import workloads
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29600 + (os.getpid() % 300)
    procs = [ctx.Process(target=_gloo_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    wl = workloads.make_workload(1, npv=101, npt=50)
    (r0, b0, e0, t0, n0, s0), (r1, b1, e1, t1, n1, s1) = res
    assert (b0, e0, b1, e1) == (0, 51, 51, 101)
    assert t0 == t1 == 11.0
    assert n0 == n1 == float(wl.evaluations)
    assert abs((s0 + s1) - wl.pv[:, 0].sum()) < 1e-12


def test_bench_reference_arm_runs_on_cpu():
    """bench.py --impl reference: the oracle on the host cores, one JSON line."""
    import json
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference",
                          "--steps", "1", "--warmup", "0", "--config", "1", "--npv", "8",
                          "--npt", "500"], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0


def test_binding_refuses_unknown_handles_and_wrong_sizes_without_a_device():
    """The wrappers check dtype and element counts against what rr_create / rr_set_data were told
    before any pointer reaches the library (the C side sees raw pointers only)."""
    import paper_2009_08500_b200 as rr
    with pytest.raises(ValueError, match="unknown ctx"):
        rr.rr_evaluate_host(123456, np.ones((1, 1, 100)), np.ones((1, 7)), np.ones((1, 10)))
    rr._CTX[999] = dict(precision=rr.RR_FP32, nz=100, ng=100, nk=50, npb=1, nkpb=1, npt=10, npv=0)
    try:
        pv = np.ones((2, 7))
        with pytest.raises(TypeError, match="float32"):       # fp64 profile for an fp32 ctx
            rr.rr_evaluate_host(999, np.ones((2, 1, 100)), pv, np.ones((2, 10), np.float32))
        with pytest.raises(ValueError, match="flux"):         # short flux buffer
            rr.rr_evaluate_host(999, np.ones((2, 1, 100), np.float32), pv,
                                np.ones((2, 9), np.float32))
        with pytest.raises(ValueError, match="ldp"):          # profile of another resolution
            rr.rr_evaluate_host(999, np.ones((2, 1, 50), np.float32), pv,
                                np.ones((2, 10), np.float32))
        with pytest.raises(TypeError, match="status"):
            rr.rr_evaluate_host(999, np.ones((2, 1, 100), np.float32), pv,
                                np.ones((2, 10), np.float32), np.zeros(2, np.int64))
    finally:
        rr._CTX.pop(999)


def test_workload_4b_is_config_4_with_literal_cadence():
    """SURVEY 8(d)'s labelled secondary workload: same population and LD draws as config 4, 10^5
    exposures spaced two minutes apart (centred on t = 0)."""
    import workloads
    a = workloads.make_workload(4, npv=5, npt=1001)
    b = workloads.make_workload("4b", npv=5, npt=1001)
    assert b.name == "config4b-literal-cadence" and a.name == "config4-stress"
    assert np.array_equal(a.pv, b.pv) and np.array_equal(a.ld_coeffs, b.ld_coeffs)
    assert np.allclose(np.diff(b.times), 2.0 / 1440.0, rtol=0, atol=1e-15)
    assert abs(b.times[500]) < 1e-15 and b.evaluations == a.evaluations


def test_bench_reference_arm_takes_the_secondary_workload():
    import json
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference",
                          "--steps", "1", "--warmup", "0", "--config", "4b", "--npv", "4",
                          "--npt", "700"], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["config"]["workload"] == "config4b-literal-cadence" and line["value"] > 0
    assert "every" in line["cpu_baseline"]["sample"] and line["cpu_baseline"]["cpu_model"]
