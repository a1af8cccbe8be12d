"""The N > 1 path of bench.py is "replicas only" (north_star fixes one GPU, no
data-path collective): each rank runs the whole workload and only the timing is reduced.  These
tests run that host-side logic with world_size 2 on the gloo backend (CPU)."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
# rank r "measured" 100 + 7 r ms over the timed steps, 50 + r ms end to end, 35 + r launches
t_max, e2e, launches = bench.reduce_over_ranks(100.0 + 7 * rank, 50.0 + rank, 35 + rank, world, "cpu")
value = bench.aggregate_value(world, 2.0e9, 5, t_max)
dist.barrier()
print(json.dumps(dict(rank=rank, world=world, t_max=t_max, e2e=e2e, launches=launches, value=value)), flush=True)
dist.destroy_process_group()
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_replica_reduction_world_size_2_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=300)
        assert p.returncode == 0, e[-2000:]
        outs.append(json.loads(o.strip().splitlines()[-1]))
    for d in outs:
        assert d["world"] == 2
        assert d["t_max"] == 107.0 and d["e2e"] == 51.0          # MAX over ranks
        assert d["launches"] == 35 + 36                          # SUM over ranks
        # whole-job value: both replicas' terms over the slower rank's time
        assert abs(d["value"] - 2 * 2.0e9 * 5 / 0.107) < 1e-3 * d["value"]
    # single rank: no process group needed
    import bench
    assert bench.reduce_over_ranks(3.0, 2.0, 7, 1, "cpu") == (3.0, 2.0, 7)


def test_reference_arm_runs_on_rank_0_only():
    """`bench.py --impl reference` under a 2-rank launch: rank 1 exits 0 without work or output."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
               MASTER_PORT=str(_free_port()))
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0", "--config", "1"], env=env, capture_output=True, text=True,
                       timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env["RANK"] = "0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0", "--config", "1", "--ref-seconds", "0.5"], env=env,
                       capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["gpu_launches"] == 0 and line["value"] > 0
