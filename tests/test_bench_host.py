"""Host-side logic of bench.py for N > 1 (replicas only, no data-path collective): the
max-over-ranks timing and the whole-job aggregate, on CPU with the gloo backend and world_size 2; the reference arm
runs on rank 0 only."""
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


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = [10.0 + 5.0 * rank, 3.0 - rank]            # rank 1 is slower on the first clock, rank 0 on the second
    got = bench.max_over_ranks(ms, dist, "cpu")
    dist.barrier()
    out.put((rank, got, bench.job_throughput(world, 256 ** 3, 20, got[0])))
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, got, value in res:
        assert got == [15.0, 3.0]                                    # the same maxima on every rank
        assert value == pytest.approx(2 * 256 ** 3 * 20 / 15.0e-3 / 1e9)   # both boxes' cells over the slowest time


def test_single_process_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([1.5, 2.5], None, "cpu") == [1.5, 2.5]
    assert bench.job_throughput(1, 1000, 2, 1.0) == pytest.approx(2e-3)


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env["RANK"] = "0"; env["LOCAL_RANK"] = "0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0", "--workload", "cfg3@32"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["n_gpus"] == 2


def test_parity_helpers_locate_where_rounding_can_act():
    """tests/parity.py: nonuniform_mask / perturb_like_fp32 / stable_entries (the conditioning protocol of reading R28)."""
    import numpy as np
    import parity as PT
    gas = np.ones((5, 16, 16, 16), dtype=np.float32)
    gas[2, 8, 8, 8] = 2.0                                     # one cell differs
    m = PT.nonuniform_mask(gas, reach=4)
    assert m[8, 8, 8] and m[8, 8, 4] and m[8, 8, 12] and m[4, 8, 8] and m[8, 12, 8]
    assert not m[8, 8, 3] and not m[8, 8, 13] and not m[0, 0, 0] and not m[9, 9, 8]
    assert m.sum() == 1 + 3 * 8                               # the cell and 4 cells either side along each axis
    p = PT.perturb_like_fp32(gas, 1)
    assert np.array_equal(p[:, ~m], gas[:, ~m].astype(np.float64))          # exactly uniform surroundings stay exact
    assert np.all(np.abs(p[:, m] / gas[:, m] - 1) < 1e-6) and np.any(p[:, m] != gas[:, m])
    ref = np.array([1.0, 2.0, -3.0, 0.0])
    ok = PT.stable_entries(ref, [ref + np.array([0, 1e-7, 0, 1e-3]), ref + np.array([1e-9, 0, 0.5, 0])], tol=1e-5)
    assert ok.tolist() == [True, True, False, False]
    e_max, e_l2 = PT.masked_errors(ref + 1e-6, ref, ok)
    assert abs(e_max - 1e-6 / 3.0) < 1e-12
