"""Host logic of bench.py under a multi-process launch (no GPU): the path does not shard
("replicas only"), so N ranks run N independent replicas and torch.distributed carries
only the barrier and the max over ranks of the device time.  Here: world_size 2 on CPU."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _torchrun(args, port):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(port)] + args
    return subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=600)


def test_reference_arm_two_ranks_prints_one_line():
    """--impl reference under torchrun: rank 0 alone runs the oracle sample and prints ONE JSON line,
    the other rank exits 0 without work."""
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--config", "1"], 29731)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    rec = json.loads(lines[0])
    assert rec["impl"] == "reference" and rec["n_gpus"] == 2 and rec["value"] > 0
    assert rec["cpu_baseline"]["kind"] == "oracle" and rec["e2e"]["h2d_bytes_per_step"] == 0


def test_max_over_ranks_and_barrier_gloo(tmp_path):
    """bench.py's own timing helpers (rank_barrier, rank_max: a barrier, then all_reduce MAX of the device
    time) on gloo, world_size 2: every rank must see the slower rank's time."""
    script = tmp_path / "w.py"
    script.write_text(
        "import sys, torch.distributed as dist\n"
        f"sys.path.insert(0, {ROOT!r})\n"
        "import bench\n"
        "dist.init_process_group('gloo')\n"
        "rank = dist.get_rank()\n"
        "synced = []\n"
        "bench.rank_barrier(dist, lambda: synced.append(1))\n"
        "assert synced == [1]\n"
        "t = bench.rank_max(dist, 10.0 + 5.0 * rank)\n"
        "assert t == 15.0, t\n"
        "assert bench.rank_max(None, 7.5) == 7.5\n"
        "if rank == 0: print('MAX', t)\n"
        "dist.destroy_process_group()\n")
    r = _torchrun([str(script)], 29732)
    assert r.returncode == 0, r.stderr[-2000:]
    assert "MAX 15.0" in r.stdout
