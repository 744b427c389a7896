"""N > 1 host logic on CPU (gloo, world_size 2).  The path is "replicas only" (SURVEY.md 8(e):
single GPU, no data-path collective), so what N > 1 adds is bench.py's rank plumbing: the
barrier, time = MAX over ranks, tokens = SUM over ranks, and the reference arm running on rank
0 only.  These run here without a GPU."""
import json
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _spawn(code, world=2, extra_env=None):
    port = _free_port()
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(world),
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), PYTHONPATH=ROOT)
        env.update(extra_env or {})
        procs.append(subprocess.Popen([sys.executable, "-c", code], env=env, cwd=ROOT,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=180)
        assert p.returncode == 0, e[-2000:]
        outs.append(o)
    return outs


def test_aggregate_is_max_time_and_sum_tokens_over_ranks():
    code = textwrap.dedent("""
        import bench, json
        rank, world = bench.init_dist("gloo")
        bench.barrier(world)
        ms, tok = bench.aggregate(10.0 + 5.0 * rank, 1000 + rank, world)
        bench.barrier(world)
        print(json.dumps({"rank": rank, "world": world, "ms": ms, "tok": tok}))
    """)
    outs = [json.loads(o.strip().splitlines()[-1]) for o in _spawn(code)]
    assert sorted(o["rank"] for o in outs) == [0, 1]
    for o in outs:
        assert o["world"] == 2
        assert o["ms"] == 15.0            # MAX over ranks
        assert o["tok"] == 2001           # SUM over ranks


def test_reference_arm_runs_on_rank0_only():
    """bench.py --impl reference under a 2-rank launch: rank 0 prints the one JSON line, the
    other rank exits 0 without work (and without needing a process group)."""
    port = _free_port()
    outs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference",
                            "--gpus", "2", "--steps", "1", "--warmup", "1", "--config", "0"],
                           env=env, cwd=ROOT, capture_output=True, text=True, timeout=300)
        assert p.returncode == 0, p.stderr[-2000:]
        outs.append(p.stdout.strip())
    assert outs[1] == ""
    line = json.loads(outs[0].splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2
    assert line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["gpu_launches"] == 0
