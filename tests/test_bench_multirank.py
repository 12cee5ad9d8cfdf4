"""bench.py's N > 1 logic on CPU: two gloo ranks reduce their times (MAX) and work counts (SUM) with the
same functions the GPU arm uses, and the headline arithmetic treats ranks as replicas (weak scaling)."""
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, %r)
    import torch.distributed as dist
    import bench
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    # rank r took (100 + 10 r) ms for 2 steps and traced (1000 + r) attempts, (800 + r) accepts per step
    times, counts = bench.reduce_over_ranks(dist, "cpu", [100.0 + 10.0 * rank, 0.5 + rank], [1000 + rank, 800 + rank, 64, 2])
    head = bench.headline(times[0], 2, counts[0], counts[1], world)
    if rank == 0:
        print(json.dumps({"times": times, "counts": counts, "head": head, "world": world}))
    dist.destroy_process_group()
""") % ROOT


def test_two_gloo_ranks_reduce_max_time_and_sum_work(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                          "--master-addr", "127.0.0.1", "--master-port", "29653", str(script)],
                         capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    import json
    line = [ln for ln in out.stdout.splitlines() if ln.startswith("{")][-1]
    d = json.loads(line)
    assert d["world"] == 2
    assert d["times"] == [110.0, 1.5]                       # MAX over ranks
    assert d["counts"] == [2001.0, 1601.0, 128.0, 4.0]      # SUM over ranks
    h = d["head"]
    assert abs(h["ms_per_step"] - 55.0) < 1e-12
    assert abs(h["value"] - 55.0e6 / 2001.0) < 1e-6         # ns per photon per attempted step, whole job
    assert abs(h["images_per_s"] - 2 / 0.055) < 1e-9        # two replicas, one image each per step


def test_single_process_path_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    times, counts = bench.reduce_over_ranks(None, "cpu", [3.0], [7, 5])
    assert times == [3.0] and counts == [7.0, 5.0]


def test_reference_arm_runs_on_rank0_only(tmp_path):
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0", "--cpu-sample", "16"], capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0 and out.stdout.strip() == ""
    env["RANK"] = "0"
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0", "--cpu-sample", "16"], capture_output=True, text=True, env=env, timeout=300)
    import json
    d = json.loads(out.stdout.strip().splitlines()[-1])
    assert d["impl"] == "reference" and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["higher_is_better"] is False
