"""Host logic of bench.py on CPU: the max-over-ranks aggregation over a world-size-2 gloo group (the N > 1 path is
"replicas only": no data-path collective), the clock summary, the roofline denominators and
the reference arm's JSON line."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def _worker(rank, world, port, q):
    import torch.distributed as dist
    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    ms, updates = bench.aggregate_over_ranks(10.0 + 5.0 * rank, 1000 * (rank + 1), dist)
    q.put((rank, ms, updates))
    dist.destroy_process_group()


def test_aggregate_over_two_gloo_ranks_takes_max_time_and_summed_work():
    torch = pytest.importorskip("torch")
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for _, ms, updates in res:
        assert ms == 15.0            # max over ranks
        assert updates == 3000.0     # whole-job work


def test_aggregate_single_process_is_identity():
    assert bench.aggregate_over_ranks(3.5, 42) == (3.5, 42)


def test_clock_summary_median_and_reasons():
    rows = [["1965", "1965", "700.1", "Not Active", "Not Active", "Not Active", "Not Active"],
            ["1400", "1965", "990.0", "Not Active", "Not Active", "Not Active", "Active"],
            ["1500", "1965", "980.0", "Not Active", "Not Active", "Not Active", "Active"],
            ["garbage"]]
    s = bench.summarize_clocks(rows)
    assert s["sm_mhz"] == 1500.0 and s["sm_max_mhz"] == 1965.0 and s["reasons"] == ["sw_power_cap"] and s["samples"] == 3
    assert bench.summarize_clocks([])["samples"] == 0


def test_roofline_denominator_and_bytes_per_update():
    peak, src = bench.measured_peak_gbs()
    assert peak > 1000.0 and ("measured" in src or "fallback" in src)
    assert bench.BYTES_PER_UPDATE == {"f64": 72.0, "f32": 36.0}      # read xi + read b + write xi', 3 components each
    t = bench.recorded_traffic("C4", "sym_tmem_f64")
    assert t is None or 0.9 < t / (72.0 * 256 * 256 * 512) < 1.5


def test_traffic_rows_of_other_sources_are_never_printed(tmp_path, monkeypatch):
    """roofline.traffic comes from a committed ncu capture; a row taken with other CUDA sources must not be quoted."""
    fp = bench.csrc_fingerprint()
    assert len(fp) == 16 and fp == bench.csrc_fingerprint()
    prof = tmp_path / "profiles"
    prof.mkdir()
    (prof / "traffic.csv").write_text("workload,kernel,dram_bytes_per_launch,csrc_sha1,source\n"
                                      "C4,sym_tmem_f64,2400000000,0123456789abcdef,stale\n"
                                      "C4,direct_tma_f64,2410000000,%s,fresh\n" % fp)
    monkeypatch.setattr(bench, "ROOT", str(tmp_path))
    monkeypatch.setattr(bench, "csrc_fingerprint", lambda: fp)
    assert bench.recorded_traffic("C4", "sym_tmem_f64") is None
    assert bench.recorded_traffic("C4", "direct_tma_f64") == 2410000000.0


def test_gpus_flag_must_match_the_launch():
    """--gpus N without N launched ranks must fail instead of printing n_gpus: 1 (run plain, WORLD_SIZE is 1)."""
    env = dict(os.environ, WORLD_SIZE="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "8", "--steps", "1"], capture_output=True, text=True,
                         timeout=300, cwd=ROOT, env=env)
    assert out.returncode != 0 and "WORLD_SIZE" in (out.stderr + out.stdout)


def test_reference_arm_prints_one_json_line_on_cpu():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "1"],
                         capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "updates/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
