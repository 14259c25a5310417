"""The N > 1 path of bench.py on CPU (world_size 2, gloo, 127.0.0.1).  The hot path does not shard (DESIGN.md 8:
"replicas only", no data-path collective), so what N > 1 adds is host logic only: the barrier, the max-over-ranks of the
device time, the whole-job value, and "rank 0 alone prints".  These tests run that logic without a GPU."""
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
    port = s.getsockname()[1]
    s.close()
    return port


def _spawn(code, world, extra_env=None):
    port = _free_port()
    procs = []
    for rank in range(world):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), **(extra_env or {}))
        procs.append(subprocess.Popen([sys.executable, "-c", code], env=env, cwd=ROOT, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=300) for p in procs]
    return [(p.returncode, o, e) for p, (o, e) in zip(procs, outs)]


def test_max_over_ranks_and_job_value_gloo():
    code = textwrap.dedent("""
        import os, sys, json
        sys.path.insert(0, %r)
        import torch, torch.distributed as dist
        import bench
        dist.init_process_group("gloo")
        rank, world = dist.get_rank(), dist.get_world_size()
        dist.barrier()
        ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist, "cpu")       # rank 1 is the slow replica
        val = bench.whole_job_tflops(world, 2.0e12, ms / 10)             # 10 steps of 2 TFLOP each
        print(json.dumps({"rank": rank, "ms": ms, "value": val}))
        dist.destroy_process_group()
    """) % ROOT
    res = _spawn(code, 2)
    for rc, out, err in res:
        assert rc == 0, err[-2000:]
    got = [json.loads(out.strip().splitlines()[-1]) for _, out, _ in res]
    for g in got:
        assert g["ms"] == 15.0                                  # every rank sees the slowest rank's time
        assert abs(g["value"] - 2 * 2.0e12 / 1.5e-3 / 1e12) < 1e-9   # 2 replicas x 2 TFLOP per step / 1.5 ms per step


def test_single_process_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.25, None, "cpu") == 3.25
    assert abs(bench.whole_job_tflops(1, 295.7e9, 0.8583) - 295.7e9 / 0.8583e-3 / 1e12) < 1e-9


def test_reference_arm_rank0_alone_prints():
    """`bench.py --impl reference` under a 2-rank launch: rank 0 times the oracle and prints the JSON line, the other
    rank exits 0 without work or output."""
    code = "import runpy, sys; sys.argv = ['bench.py', '--impl', 'reference', '--gpus', '2', '--steps', '1', '--warmup', '0']; runpy.run_path('bench.py', run_name='__main__')"
    res = _spawn(code, 2)
    (rc0, out0, err0), (rc1, out1, err1) = res
    assert rc0 == 0, err0[-2000:]
    assert rc1 == 0, err1[-2000:]
    assert out1.strip() == ""
    line = json.loads(out0.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["metric"] == "sparse_layer_fwd_bwd_tflops_670k" and line["higher_is_better"] is True
