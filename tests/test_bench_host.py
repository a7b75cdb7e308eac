"""Host logic of bench.py without a GPU: work formulas, the multi-rank (replica) timing reduction on gloo with
world_size 2, and the --impl reference arm."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_work_formulas():
    import bench
    import workloads as W
    b3 = W.config3_prefill()
    assert abs(bench.prefill_flops(b3) - 0.14316e12) < 1e8          # 0.1432 TFLOP for this draw
    assert bench.append_bytes(b3) == 2 * 16777216                  # 16.8 MB in + 16.8 MB out
    b1 = W.config1_tiny_decode()
    kv, tot = bench.decode_bytes(b1, 1)
    assert kv == 77312 and tot == kv + 2 * 4 * 8 * 64 * 2 + 4 * 13 + 16


_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch, bench
rank, world, local, dist = bench.dist_setup(2)
assert world == 2 and dist is not None
dev = torch.device("cpu")
t = bench.max_over_ranks(dist, 1.5 if rank == 0 else 4.25, dev)
s = bench.sum_over_ranks(dist, 10.0 + rank, dev)
dist.barrier()
print("RESULT", rank, t, s, flush=True)
dist.destroy_process_group()
"""


def test_replica_timing_reduction_gloo_world2(tmp_path):
    """N > 1 is N independent replicas: time = max over ranks, work = sum over ranks."""
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT))
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=180)[0] for p in procs]
    for p, o in zip(procs, outs):
        assert p.returncode == 0, o
    for o in outs:
        line = [l for l in o.splitlines() if l.startswith("RESULT")][0].split()
        assert float(line[2]) == 4.25 and float(line[3]) == 21.0


def test_reference_arm_prints_contract_line():
    env = dict(os.environ, CUDA_VISIBLE_DEVICES="")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0"], env=env, capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "GB/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    # ranks other than 0 print nothing and exit 0
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference"],
                         env=dict(env, RANK="1", WORLD_SIZE="2"), capture_output=True, text=True, timeout=60)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_gpus_flag_respawns_under_torchrun(monkeypatch):
    """`python bench.py --gpus N` without torchrun becomes N ranks (one per GPU) on this node; under torchrun
    (WORLD_SIZE set) it runs as the rank it is."""
    import bench
    cmd = bench.torchrun_command(4, ["--gpus", "4", "--steps", "3"], port=29999)
    assert cmd[1:3] == ["-m", "torch.distributed.run"] and "--nproc-per-node" in cmd
    assert cmd[cmd.index("--nproc-per-node") + 1] == "4" and cmd[cmd.index("--master-addr") + 1] == "127.0.0.1"
    assert cmd[-5:] == [os.path.join(ROOT, "bench.py"), "--gpus", "4", "--steps", "3"]
    seen = {}
    monkeypatch.delenv("WORLD_SIZE", raising=False)
    monkeypatch.setattr(bench, "respawn_under_torchrun", lambda n, argv: seen.update(n=n, argv=argv) or 0)
    monkeypatch.setattr(bench, "run_ours", lambda args: seen.update(direct=args.gpus) or 0)
    assert bench.main(["--gpus", "2", "--steps", "1"]) == 0 and seen == {"n": 2, "argv": ["--gpus", "2", "--steps", "1"]}
    seen.clear()
    monkeypatch.setenv("WORLD_SIZE", "2")
    assert bench.main(["--gpus", "2"]) == 0 and seen == {"direct": 2}
    seen.clear()
    monkeypatch.delenv("WORLD_SIZE")
    assert bench.main(["--gpus", "1"]) == 0 and seen == {"direct": 1}


def test_ncu_traffic_is_read_from_the_committed_summary(tmp_path):
    import bench
    f = tmp_path / "s.csv"
    f.write_text('Kernel Name,gpu__time_duration.sum,dram__bytes_read.sum,dram__bytes_write.sum\n,us,Gbyte,Mbyte\n'
                 '"void prefill_umma_kernel<16, 0>(X)",1,0.5,2\n'
                 '"void decode_splitk_kernel<128, 32, 8, 0, 4, 1>(X)",1,2,1\n"void decode_combine_kernel<128>(X)",1,0.004,0\n')
    t = bench.load_ncu_traffic(str(f))
    assert t["prefill"] == 502000000 and t["decode"] == 2005000000
    assert bench.load_ncu_traffic(str(tmp_path / "missing.csv"))["decode"] is None
