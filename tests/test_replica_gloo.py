"""N > 1 host logic on CPU: two gloo ranks, max-over-ranks timing and the frame split (replicas only)."""
import os
import socket

import torch.multiprocessing as mp


def _worker(rank, world, port, q):
    import torch.distributed as dist
    from paper_2407_10707_b200 import replica
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    fps, ms = replica.whole_job_fps(2.0 if rank == 0 else 4.0, world)
    frames = list(replica.frames_of_rank(7, rank, world))
    q.put((rank, fps, ms, frames))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_gloo_timing_and_split():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    out = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    # slowest rank (4 ms/step) sets the job time; 2 ranks x 1 frame per step -> 500 frames/s on both ranks
    assert all(abs(o[1] - 500.0) < 1e-9 and abs(o[2] - 4.0) < 1e-12 for o in out)
    assert out[0][3] == [0, 1, 2, 3] and out[1][3] == [4, 5, 6]


def test_single_process_passthrough():
    from paper_2407_10707_b200 import replica
    assert replica.max_over_ranks([1.5, 2.5]) == [1.5, 2.5]
    assert list(replica.frames_of_rank(64, 3, 8)) == list(range(24, 32))
