"""CPU checks of bench.py's multi-rank plumbing (world_size 2, gloo) and of its reference arm."""
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
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, "cpu")          # rank 1 is the slow one
    out.put((rank, ms, bench.whole_job_value(1_000_000_000, 4, world, ms)))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_world2_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [15.0, 15.0]                           # both see the max
    # 2 replicas x 4 steps x 1 GB in 15 ms
    assert res[0][2] == pytest.approx(2 * 4 * 1e9 / 15e-3 / 1e9)


def test_single_rank_helpers_do_not_need_a_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, 1, "cpu") == 3.5
    assert bench.whole_job_value(2_000_000_000, 10, 1, 100.0) == pytest.approx(200.0)


def test_reference_arm_under_torchrun_rank0_prints_one_line():
    env = dict(os.environ, OMP_NUM_THREADS="4")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(29600 + os.getpid() % 300), os.path.join(ROOT, "bench.py"),
           "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["value"] > 0 and d["unit"] == "GB/s"


def test_reference_arm_without_torchrun_reports_the_gpu_count_it_was_given():
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    env["OMP_NUM_THREADS"] = "4"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0"], capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0


def test_bare_gpus_n_starts_n_ranks_itself(monkeypatch):
    """`python bench.py --gpus 2` with WORLD_SIZE unset re-executes itself under torch.distributed.run with 2 ranks."""
    sys.path.insert(0, ROOT)
    import bench
    seen = {}

    def fake_execv(exe, argv):
        seen["argv"] = argv
        raise SystemExit(0)
    monkeypatch.setattr(bench.os, "execv", fake_execv)
    monkeypatch.setattr(sys, "argv", ["bench.py", "--gpus", "2", "--steps", "3"])
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        monkeypatch.delenv(k, raising=False)
    with pytest.raises(SystemExit):
        bench.main()
    argv = seen["argv"]
    assert "torch.distributed.run" in argv and "--nproc-per-node=2" in argv and "127.0.0.1" in argv
    assert argv[-4:] == ["--gpus", "2", "--steps", "3"] and argv[-5].endswith("bench.py")


def test_ncu_traffic_is_reported_only_for_the_tree_it_was_captured_on(tmp_path, monkeypatch):
    """roofline.traffic comes from a committed ncu capture keyed by the hash of the kernel sources: a capture taken
    on other sources reads as null (with a note), never as a number."""
    sys.path.insert(0, ROOT)
    import bench
    f = tmp_path / "ncu_traffic.json"
    monkeypatch.setattr(bench, "NCU_TRAFFIC_FILE", str(f))
    assert bench.ncu_traffic()[0] is None                                  # no file
    f.write_text(json.dumps({"kernel_source_sha256": bench.kernel_source_hash(), "step_kernel_dram_bytes_per_launch": 123, "capture": "x"}))
    assert bench.ncu_traffic()[0] == 123
    f.write_text(json.dumps({"kernel_source_sha256": "0" * 64, "step_kernel_dram_bytes_per_launch": 123, "capture": "x"}))
    val, note = bench.ncu_traffic()
    assert val is None and "stale" in note
