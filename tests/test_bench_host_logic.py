"""Host-side logic of bench.py without a GPU: the multi-rank aggregation (world_size 2, gloo),
the reference arm, and the layout arithmetic shared with DESIGN.md."""
import json
import os
import subprocess
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=int(sys.argv[1]), world_size=2)
rank = dist.get_rank()
# rank 0 did 10 products in 5 ms, rank 1 did 10 products in 8 ms -> 20 products / 8 ms
value, ms = bench.aggregate_throughput(10.0, 5.0 if rank == 0 else 8.0, 2)
mx = bench.max_over_ranks(float(rank), 2)
dist.barrier()
dist.destroy_process_group()
print(json.dumps({{"rank": rank, "value": value, "ms": ms, "mx": mx}}))
"""


def test_aggregate_over_two_ranks_gloo(tmp_path):
    port = 29500 + (os.getpid() % 2000)
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=str(ROOT), port=port))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, text=True)
             for r in range(2)]
    outs = [p.communicate(timeout=120)[0] for p in procs]
    assert all(p.returncode == 0 for p in procs)
    for out in outs:
        d = json.loads(out.strip().splitlines()[-1])
        assert d["ms"] == 8.0
        assert d["value"] == pytest.approx(20.0 / 8e-3)
        assert d["mx"] == 1.0


def test_single_rank_aggregate_is_identity():
    sys.path.insert(0, str(ROOT))
    import bench
    value, ms = bench.aggregate_throughput(7.0, 3.5, 1)
    assert ms == 3.5 and value == pytest.approx(2000.0)
    assert bench.transform_length(7) == 16 and bench.transform_length(63) == 128
    assert bench.transform_length(0) == 1 and bench.transform_length(8) == 32 and bench.transform_length(127) == 256
    # products of the series exponential: Horner below N_trunc = 6, Paterson-Stockmeyer above
    assert [bench.exp_products(n) for n in (0, 1, 5, 6, 31, 63, 127)] == [0, 0, 4, 4, 10, 14, 21]


def test_reference_arm_prints_one_json_line():
    out = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--workload", "small",
                          "--steps", "2", "--warmup", "1"], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle"
    assert line["value"] > 0 and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["higher_is_better"] is True and line["unit"] == "products/s"


def test_reference_arm_nonzero_rank_exits_quietly():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--workload", "small",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=120, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_reference_arm_uses_the_cuda_arm_workload_string():
    sys.path.insert(0, str(ROOT))
    import bench
    out = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--workload", "small",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=120)
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["config"]["workload"] == bench.WORKLOAD_DESC["small"]
    assert "1 full star-product" in line["cpu_baseline"]["sample"]


def test_replica_environment_and_cpu_fftconv():
    sys.path.insert(0, str(ROOT))
    import numpy as np
    import bench
    import oracle
    from paper_2001_02835_b200 import workloads as wl
    env = bench.replica_env(3, 4, 12345)
    assert (env["RANK"], env["LOCAL_RANK"], env["WORLD_SIZE"], env["MASTER_ADDR"], env["MASTER_PORT"]) == \
        ("3", "3", "4", "127.0.0.1", "12345")
    # the second CPU baseline (the paper's FFT-CONV with library FFT + GEMM) computes the same product as the oracle
    A, B = wl.config_product(12, 9, seed=[7, 12, 9])
    err = oracle.per_order_error(bench.cpu_fftconv(A, B), oracle.series_mul(A, B), oracle.product_bound(A, B)).max()
    assert err < 1e-13
