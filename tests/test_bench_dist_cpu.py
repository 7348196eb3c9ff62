"""Host logic of bench.py's N > 1 path on CPU: world-size-2 gloo rendezvous on 127.0.0.1, the
max-over-ranks aggregation of the per-rank device times, and the reference arm's rank gating.
("Replicas only": the data path has no collective - DESIGN.md section 8.)"""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, os.environ["FK_ROOT"])
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ms = bench.aggregate_max(1.0 + 2.5 * rank, world)
dist.barrier()
print(json.dumps({"rank": rank, "world": world, "ms": ms}))
dist.destroy_process_group()
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_max_over_ranks_with_gloo_world_size_2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = str(_free_port())
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=port, FK_ROOT=ROOT)
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=180)
        assert p.returncode == 0, err
        outs.append(json.loads(out.strip().splitlines()[-1]))
    assert sorted(o["rank"] for o in outs) == [0, 1]
    for o in outs:
        assert o["world"] == 2 and o["ms"] == 3.5   # the slower rank's time, on every rank


def test_single_rank_aggregate_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate_max(1.25, 1) == 1.25


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert p.returncode == 0 and p.stdout.strip() == ""


def test_step_bytes_counts_two_table_reads():
    sys.path.insert(0, ROOT)
    import bench
    from paper_1909_10547_b200 import synth
    case = synth.hadronic_case(6, 4, 5, 3, 1, sub=9)
    b = bench.step_bytes(case)
    assert b == 2 * case.fk.nbytes + 3 * case.f.nbytes + 2 * case.N * 8


def test_gpus_n_fails_loudly_without_n_devices():
    """`python bench.py --gpus 2` must never print an N=1 line: without a torchrun environment it spawns the ranks
    itself, and on a node with fewer than 2 GPUs (this CPU box: 0) it refuses."""
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1", "--warmup", "0"],
                       env=env, capture_output=True, text=True, timeout=180)
    assert p.returncode != 0
    assert p.stdout.strip() == ""
    assert "--gpus 2" in p.stderr and "refusing" in p.stderr


def test_world_size_must_match_gpus_flag():
    env = dict(os.environ, RANK="0", LOCAL_RANK="0", WORLD_SIZE="4")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1", "--warmup", "0"],
                       env=env, capture_output=True, text=True, timeout=180)
    assert p.returncode != 0 and "WORLD_SIZE=4" in p.stderr


def test_reference_arm_reports_one_gpu():
    """The reference arm runs on rank 0's host cores: its line says n_gpus 1 whatever --gpus is."""
    env = dict(os.environ, RANK="0", WORLD_SIZE="2", OMP_NUM_THREADS="4")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=600)
    assert p.returncode == 0, p.stderr
    line = json.loads(p.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 1 and line["value"] > 0
