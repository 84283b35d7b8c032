"""N > 1 plumbing of bench.py on CPU (gloo, world_size 2): the path is "replicas only",
so what needs covering is the launch contract: RANK / WORLD_SIZE / LOCAL_RANK parsing, max-over-ranks
time, sum-over-ranks work, rank 0 alone printing, and the reference arm under torchrun."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def torchrun(args, nproc=2, timeout=600):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={nproc}",
           "--master-addr", "127.0.0.1", "--master-port", str(free_port())] + args
    env = dict(os.environ, OMP_NUM_THREADS="2", CUDA_VISIBLE_DEVICES="")
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def json_lines(out):
    return [json.loads(ln) for ln in out.splitlines() if ln.startswith("{")]


def test_aggregation_over_two_gloo_ranks():
    r = torchrun([os.path.join(ROOT, "tests", "_multirank_worker.py")])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = json_lines(r.stdout)
    assert len(lines) == 1                                  # rank 0 alone prints
    assert lines[0] == {"ms": 11.0, "updates": 3000.0, "world": 2, "local": 0}


def test_reference_arm_under_torchrun_prints_one_line():
    r = torchrun([os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--config", "1",
                  "--steps", "2", "--warmup", "1"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = json_lines(r.stdout)
    assert len(lines) == 1
    d = lines[0]
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["unit"] == "unknown-updates/s"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"] > 0
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["iters_per_step"] == [7, 7]                    # config 1, oracle (tests/golden)


def test_single_process_aggregation_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate_over_ranks(None, 3.5, 7.0, None) == (3.5, 7.0)
    assert bench.dist_env() == (int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1)),
                                int(os.environ.get("LOCAL_RANK", 0)))
