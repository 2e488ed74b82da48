"""N > 1 path on CPU: two `gloo` ranks run the host logic of `bench.py --gpus 2` ("replicas only").

The tracker shards by independent time frames, so the only exchange is the reduction of the timing: job time = MAX
over ranks, job work = SUM of the clusters the ranks tracked.  No GPU, no tracker arithmetic here.
"""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2102_08862_b200 import gen, replicas


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert replicas.rank_world_local() == (rank, world, rank)
        # each rank generates its own (small) frame, as bench.py does with seed + rank
        cfg = gen.preset(0, replicas.frame_seed(11, rank))
        tf = gen.generate(cfg, want_truth=False)
        # a made-up device time per rank: rank 1 is the slow one
        total_ms = 40.0 + 25.0 * rank
        steps = 5
        ms_per_step, value, n_all = replicas.aggregate(total_ms, tf.n, steps, world)
        e2e_ms = replicas.max_over_ranks(3.0 + rank, world)
        torch.save({"n": tf.n, "ms_per_step": ms_per_step, "value": value, "n_all": n_all, "e2e_ms": e2e_ms,
                    "row_head": torch.from_numpy(tf.row[:64].copy())}, os.path.join(out_dir, f"r{rank}.pt"))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_two_gloo_ranks_track_different_frames_and_agree_on_the_job_numbers(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    r = [torch.load(os.path.join(str(tmp_path), f"r{k}.pt")) for k in range(world)]
    # different frames per rank (seed + rank), same generator
    assert r[0]["n"] > 1000 and r[1]["n"] > 1000
    assert r[0]["n"] != r[1]["n"] or not torch.equal(r[0]["row_head"], r[1]["row_head"])
    # every rank holds the same whole-job numbers
    for key in ("ms_per_step", "value", "n_all", "e2e_ms"):
        assert r[0][key] == r[1][key], key
    # time = max over ranks, work = sum over ranks
    assert r[0]["ms_per_step"] == pytest.approx(65.0 / 5)
    assert r[0]["n_all"] == r[0]["n"] + r[1]["n"]
    assert r[0]["value"] == pytest.approx((r[0]["n"] + r[1]["n"]) / (13.0e-3))
    assert r[0]["e2e_ms"] == 4.0


def test_single_rank_aggregate_needs_no_process_group():
    ms, value, n_all = replicas.aggregate(50.0, 1000, 10, 1)
    assert (ms, value, n_all) == (5.0, 1000 / 5.0e-3, 1000.0)
    assert replicas.max_over_ranks(7.5, 1) == 7.5
    assert replicas.frame_seed(3, 4) == 7
    with pytest.raises(ValueError):
        replicas.aggregate(1.0, 1, 0, 1)
    with pytest.raises(RuntimeError):
        replicas.aggregate(1.0, 1, 1, 2)
