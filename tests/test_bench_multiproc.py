"""The N > 1 host logic of bench.py on CPU (gloo, world_size 2): the path does not shard (DESIGN.md "Multi-GPU":
replicas only), so all that ranks exchange is the timing -- max over ranks -- and rank 0 alone prints the line."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist, "cpu")  # rank 1 is the slow one
    q.put((rank, ms, bench.aggregate_value(world, 1000, 4, ms)))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [g[1] for g in got] == [15.0, 15.0]                      # both ranks see the slowest rank's time
    assert got[0][2] == pytest.approx(2 * 1000 * 4 / 15e-3)         # two replicas' cells over that time


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, None, "cpu") == 3.5
    assert bench.aggregate_value(1, 10, 2, 1000.0) == pytest.approx(20.0)


def test_reference_arm_under_torchrun_prints_one_line():
    """`--impl reference` launched like the driver launches N = 2: rank 0 times the oracle, rank 1 exits 0 silently."""
    env = dict(os.environ, OMP_NUM_THREADS="1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"), "--impl", "reference",
           "--gpus", "2", "--steps", "1", "--warmup", "0", "--config", "1"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0


def test_algorithmic_bytes_and_committed_traffic():
    """B_alg per cell-step = 2128 B (configs 1, 2), 2176 B (3, 5), 3040 B (4); and the ncu traffic file that
    bench.py's roofline.traffic reads carries both kernel classes, above their algorithmic bytes."""
    sys.path.insert(0, ROOT)
    import bench
    from paper_2412_04395_b200 import workloads as wl
    want = {1: 2128, 2: 2128, 3: 2176, 4: 3040, 5: 2176}
    for cfg, b in want.items():
        case = wl.make_case(cfg, nx=8, ny=8, with_state=False)
        assert bench.algorithmic_doubles(case)["total"] * 8 == b, cfg
    cells = 1024 * 1024 * 128
    ac, sl = bench.measured_traffic("acoustic_fused", 5), bench.measured_traffic("slow_rhs_fused", 5)
    assert ac is not None and sl is not None
    assert 20 * 8 * cells < ac < 2.0 * 20 * 8 * cells
    assert 14 * 8 * cells < sl < 4.0 * 14 * 8 * cells
    assert bench.measured_traffic("acoustic_fused", 3) is None
