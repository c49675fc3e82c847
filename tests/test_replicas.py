"""The N > 1 path of bench.py is REPLICAS ONLY (north_star: one GPU, no sharding): its only communication is
the timing protocol -- a barrier on both sides of the timed region, MAX over ranks of the device time, and the
whole-job throughput = replicas / that time.  Covered here with world_size 2 on CPU (gloo)."""
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


def _spawn(code, world=2, extra_env=None):
    port = _free_port()
    procs = []
    for rank in range(world):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), PYTHONPATH=ROOT, OMP_NUM_THREADS="1")
        env.update(extra_env or {})
        procs.append(subprocess.Popen([sys.executable, "-c", textwrap.dedent(code)], env=env, cwd=ROOT,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=180) for p in procs]
    return [(p.returncode, o, e) for p, (o, e) in zip(procs, outs)]


def test_single_process_is_the_identity():
    from paper_2506_16676_b200 import replicas
    assert replicas.env_world() == (int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)),
                                    int(os.environ.get("WORLD_SIZE", 1)))
    assert replicas.max_over_ranks(1.25) == 1.25
    assert replicas.sum_over_ranks(1.25) == 1.25
    replicas.barrier()       # no process group: a no-op
    replicas.finalize()


def test_two_replicas_gloo_timing_protocol():
    code = """
        from paper_2506_16676_b200 import replicas
        rank, local_rank, world = replicas.init("gloo")
        assert world == 2 and rank == local_rank
        replicas.barrier()
        t = replicas.max_over_ranks(1.0 + rank)          # the slower replica sets the job time
        n = replicas.sum_over_ranks(1.0)
        replicas.barrier()
        print(f"{rank} {t} {n} {world / t}")
        replicas.finalize()
    """
    res = _spawn(code)
    for rank, (rc, out, err) in enumerate(res):
        assert rc == 0, err
        r, t, n, thr = out.split()
        assert int(r) == rank and float(t) == 2.0 and float(n) == 2.0 and float(thr) == 1.0


def test_reference_arm_runs_on_rank_0_only():
    """bench.py --impl reference under torchrun: rank 0 prints the line, the other ranks exit 0 without work."""
    code = """
        import sys
        sys.argv = ["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--workload", "C0",
                    "--ref-coarse-its", "5"]
        import bench
        sys.exit(bench.main())
    """
    res = _spawn(code)
    (rc0, out0, err0), (rc1, out1, err1) = res
    assert rc0 == 0, err0
    assert rc1 == 0, err1
    assert out1.strip() == ""
    import json
    line = json.loads(out0.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle"
    assert line["cpu_baseline"]["measured"]["coarse_gmres_iterations_timed"] == 5 and line["gpu_launches"] == 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["unit"] == "s"
