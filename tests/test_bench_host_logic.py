"""Host-side logic of bench.py that needs no GPU: the N>1 aggregation (replicas only: MAX over
ranks of the device time, whole-job tets/s) under gloo with world_size 2, the reference arm's
JSON line, and the oracle sample sizing."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world)  # rank 1 is the slow replica
    out.put((rank, ms, bench.whole_job_value(1000, world, ms)))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_gloo_max_over_ranks_and_whole_job_value():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, value in got:
        assert ms == 15.0                       # the slowest replica sets the time on every rank
        assert value == pytest.approx(2 * 1000 / 15e-3)


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, 1) == 3.5
    assert bench.whole_job_value(6, 1, 2.0) == pytest.approx(3000.0)


def test_sample_fraction_bounds_the_cpu_work():
    sys.path.insert(0, ROOT)
    import bench
    import psd_inputs
    for cfg in psd_inputs.CONFIGS:
        f = bench.sample_fraction(cfg)
        assert 0.0 < f <= 1.0
        assert f * 6 * cfg["N"] ** 3 <= 15e6 + 1


def test_reference_arm_prints_one_json_line_with_the_contract_keys():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference",
                        "--config", "0", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    base = json.load(open(os.path.join(ROOT, "BASELINE.json")))
    assert d["impl"] == "reference" and d["metric"] == base["metric"] and d["unit"] == "tets/s"
    assert d["higher_is_better"] is True and d["vs_baseline"] is None
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"] == {"value": d["value"], "unit": "tets/s", "h2d_bytes_per_step": 0,
                        "d2h_bytes_per_step": 0}
    assert d["config"]["workload"] == "cfg0_32_64" and d["value"] > 0


def test_reference_arm_other_ranks_exit_without_work():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference",
                        "--gpus", "2"], capture_output=True, text=True, timeout=120, env=env)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_roofline_traffic_comes_from_the_committed_capture():
    import bench
    v = bench.read_ncu_traffic("cfg1_128_256", "deposit")
    assert isinstance(v, int) and v > 100e6
    assert bench.read_ncu_traffic("no_such_workload", "deposit") is None
    # the headline workload and the patch config have captures too (sums over the record slabs and
    # over the kernels of the deposit phase)
    for w, main in (("cfg4_512_1024", "k_deposit_tiles2"), ("cfg3_256_patches", "k_deposit_tiles2"),
                    ("cfg2_256_512", "k_deposit_tiles2")):
        assert bench.read_ncu_traffic(w, "deposit") > bench.read_ncu_value(w, main) > 1e9
        assert bench.read_ncu_fp64_flops(w) > 1e11
    assert bench.read_ncu_fp64_flops("no_such_workload") is None


def test_strided_oracle_sample_covers_the_lattice():
    import bench
    r = bench.strided_ranges(512 ** 3, 2_500_000)
    assert len(r) == 64 and r[0][0] == 0 and r[-1][0] > 0.98 * 512 ** 3 * 63 / 64
    assert all(b < e <= 512 ** 3 for b, e in r) and all(r[i][1] <= r[i + 1][0] for i in range(63))
    assert sum(e - b for b, e in r) <= 2_500_000
    assert bench.strided_ranges(10, 100) == [(i, i + 1) for i in range(10)]
