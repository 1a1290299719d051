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
    """The reduction bench.py uses for its timing (all_reduce MAX after a barrier), on gloo."""
    script = tmp_path / "w.py"
    script.write_text(
        "import os, torch, torch.distributed as dist\n"
        "dist.init_process_group('gloo')\n"
        "rank = dist.get_rank()\n"
        "dist.barrier()\n"
        "t = torch.tensor([10.0 + 5.0 * rank], dtype=torch.float64)\n"
        "dist.all_reduce(t, op=dist.ReduceOp.MAX)\n"
        "assert float(t.item()) == 15.0\n"
        "if rank == 0: print('MAX', float(t.item()))\n"
        "dist.destroy_process_group()\n")
    r = _torchrun([str(script)], 29732)
    assert r.returncode == 0, r.stderr[-2000:]
    assert "MAX 15.0" in r.stdout
