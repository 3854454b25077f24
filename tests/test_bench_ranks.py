"""N > 1 path of bench.py (replicas only, no data-path collective): the cross-rank reduction and the
replica frame indices, with world_size 2 on gloo/CPU; and the reference arm under two ranks (rank 0 alone prints)."""
import json
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    ms, rays = bench.reduce_over_ranks(10.0 + 5.0 * rank, 1000.0 * (rank + 1), torch.device("cpu"), world)
    frames = [bench.replica_frame_index(i, rank, world) for i in range(4)]
    out.put((rank, ms, rays, frames))
    dist.barrier()
    dist.destroy_process_group()


def test_reduce_over_ranks_world_size_2_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, rays, frames in res:
        assert ms == 15.0            # MAX over ranks
        assert rays == 3000.0        # SUM over ranks
    all_frames = res[0][3] + res[1][3]
    assert len(set(all_frames)) == 8 and sorted(all_frames) == list(range(8))     # replicas render disjoint frames


def test_single_rank_reduction_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_over_ranks(3.5, 7.0, torch.device("cpu"), 1) == (3.5, 7.0)


def test_reference_arm_two_ranks_only_rank0_prints():
    outs = []
    for rank in (0, 1):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank))
        r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                            "--workload", "cornell"], env=env, capture_output=True, text=True, timeout=300)
        assert r.returncode == 0, r.stderr
        outs.append(r.stdout.strip())
    line = json.loads(outs[0])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
    assert outs[1] == ""
