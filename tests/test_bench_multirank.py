"""N > 1 path of bench.py on CPU: world_size 2, gloo (replicas only).

Covers (i) the max-over-ranks reduction bench.py applies to every timing and (ii) the
`--impl reference` arm under torchrun: rank 0 alone runs the oracle and prints ONE JSON line, the
other rank exits 0 without output."""
import json
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _torchrun(args, port, timeout=600):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(port)] + args
    env = dict(os.environ, OMP_NUM_THREADS="2")
    return subprocess.run(cmd, cwd=ROOT, env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE,
                          text=True, timeout=timeout)


def test_max_over_ranks_gloo_world2(tmp_path):
    script = tmp_path / "w2.py"
    script.write_text(textwrap.dedent(f"""
        import os, sys
        sys.path.insert(0, {ROOT!r})
        import torch.distributed as dist
        import bench
        dist.init_process_group("gloo")
        rank, world = dist.get_rank(), dist.get_world_size()
        got = bench.max_over_ranks(10.0 + rank, world, "cpu")
        assert world == 2 and got == 11.0, (world, got)
        print(f"rank{{rank}} ok {{got}}", flush=True)
        dist.destroy_process_group()
    """))
    out = _torchrun([str(script)], 29611)
    assert out.returncode == 0, out.stderr[-2000:]
    assert "rank0 ok 11.0" in out.stdout and "rank1 ok 11.0" in out.stdout


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    out = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                     "--config", "0"], 29612)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["unit"] == "cell-updates/s"
    assert d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0


import pytest


@pytest.mark.gpu
def test_ours_arm_two_ranks_share_one_gpu_over_gloo():
    """The N > 1 path of bench.py end to end on whatever GPUs are present: two replica ranks
    (HYDRO_BENCH_BACKEND=gloo lets them share a device; they meet only at host barriers), one
    JSON line from rank 0 with the aggregate over both."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29613", "bench.py", "--gpus", "2",
           "--config", "0", "--steps", "20", "--warmup", "3", "--e2e-steps", "1"]
    env = dict(os.environ, HYDRO_BENCH_BACKEND="gloo", OMP_NUM_THREADS="2")
    out = subprocess.run(cmd, cwd=ROOT, env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE,
                         text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["scaling"] == "weak" and d["value"] > 0
    assert d["config"]["parallelism"].startswith("2 independent replicas")
    assert d["gpu_launches"] > 0 and d["cpu_baseline"] is None
