"""Host-side logic of bench.py's N > 1 path on CPU: world_size-2 `gloo` processes.  The path is
"replicas only": the ranks exchange nothing but a barrier and the max of their timings,
and the whole-job value is the work of all ranks over the slowest rank's time.  Under torchrun the
reference arm runs on rank 0 alone."""
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
    os.environ.update({"RANK": str(rank), "WORLD_SIZE": str(world), "LOCAL_RANK": str(rank),
                       "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    sys.path.insert(0, ROOT)
    import bench
    r = bench.Ranks("gloo")
    r.barrier()
    mx = r.max_over_ranks(1.0 + rank)                 # rank 1 is the slow one: 2.0 s
    val = r.whole_job_value(100.0, 1.0 + rank)        # 2 ranks x 100 units / 2.0 s
    r.barrier()
    r.close()
    q.put((rank, mx, val))


def test_two_rank_gloo_max_timing_and_aggregate():
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
    assert [g[0] for g in got] == [0, 1]
    for _, mx, val in got:
        assert mx == 2.0
        assert val == pytest.approx(100.0)


def test_single_process_ranks_is_a_no_op():
    sys.path.insert(0, ROOT)
    env = {k: os.environ.pop(k) for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK") if k in os.environ}
    try:
        import bench
        r = bench.Ranks("gloo")
        assert r.world == 1 and r.max_over_ranks(3.5) == 3.5 and r.whole_job_value(7.0, 2.0) == 3.5
        r.close()
    finally:
        os.environ.update(env)


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_bytes_model_matches_the_papers_counts():
    # 8 links x 18 (12) reals x 4 B = 576 (384) B loaded per site in SP, the same stored
    sys.path.insert(0, ROOT)
    import bench
    from tests.helpers import paper_values
    pv = paper_values()
    assert bench.bytes_per_site_update("sp", 18) == 2 * pv["bytes_loaded_per_site_sp_18"] == 2 * 576
    assert bench.bytes_per_site_update("sp", 12) == 2 * pv["bytes_loaded_per_site_sp_12"] == 2 * 384
    # App. A flop model used for paper_gflops
    assert pv["flop_gather_landau"] + pv["flop_or_update"] + pv["flop_apply"] == pv["flop_per_site_landau_or"] == 2274
    assert pv["flop_apply"] == 3 * 8 * pv["flop_per_link_subgroup"]
    assert bench.bytes_per_site_update("dp", 18) == 2304
    assert bench.bytes_per_site_update("sp", 12, nd=3) == 576
    line = json.dumps({"ok": True})
    assert json.loads(line)["ok"]
