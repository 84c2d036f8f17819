"""N > 1 path of bench.py on CPU: two processes over gloo (127.0.0.1), no GPU.

DESIGN.md "Multi-GPU": the path does not shard (north_star: one GPU, no collectives), so `--gpus N` runs N
independent replicas; what N > 1 adds is the rank plumbing -- barrier, max-over-ranks timing, whole-job
aggregation, rank 0 alone printing -- which is what these tests drive, with the backend switched to gloo.
"""
import json
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _spawn(code, world=2, timeout=240):
    port = _free_port()
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), PYTHONPATH=ROOT, OMP_NUM_THREADS="2")
        procs.append(subprocess.Popen([sys.executable, "-c", textwrap.dedent(code)], env=env, cwd=ROOT,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=timeout)
        assert p.returncode == 0, e[-2000:]
        outs.append(o)
    return outs


def test_max_over_ranks_barrier_and_whole_job_rate_gloo_world2():
    outs = _spawn("""
        import bench
        R = bench.Ranks("gloo")
        assert R.world == 2 and R.dist is not None
        R.barrier()
        t = 1.0 + R.rank                       # rank 1 is the slow one: 2 s
        m = R.max(t)
        rate = R.whole_job_rate(1000, t)       # 2 ranks x 1000 units / 2 s
        R.barrier()
        print("%d %.6f %.6f" % (R.rank, m, rate))
        R.close()
    """)
    for r, o in enumerate(outs):
        rank, m, rate = o.split()
        assert int(rank) == r and float(m) == 2.0 and float(rate) == 1000.0


def test_world1_needs_no_process_group():
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    env["PYTHONPATH"] = ROOT
    code = "import bench; R = bench.Ranks('gloo'); assert R.dist is None and R.max(3.5) == 3.5; R.barrier(); print(R.whole_job_rate(10, 2.0))"
    out = subprocess.run([sys.executable, "-c", code], env=env, cwd=ROOT, capture_output=True, text=True, timeout=120)
    assert out.returncode == 0, out.stderr[-2000:]
    assert float(out.stdout) == 5.0


def test_reference_arm_under_two_ranks_prints_one_line_from_rank0():
    """--impl reference under a 2-rank launch: rank 0 alone runs the oracle and prints the line, rank 1 exits 0."""
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port),
                   OMP_NUM_THREADS="4")
        procs.append(subprocess.Popen([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                                       "--warmup", "0", "--workload", "minkowski_64_mc"], env=env, cwd=ROOT,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=600)
        assert p.returncode == 0, e[-2000:]
        outs.append(o.strip())
    assert outs[1] == ""
    line = json.loads(outs[0])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["unit"] == "zone-cycles/s" and line["higher_is_better"] is True
