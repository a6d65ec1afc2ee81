"""N > 1 host logic on CPU: world_size-2 gloo.  Frame shards (+ read-only halo) computed
independently by each rank reproduce the single-process oracle result bit for bit; the only
communication is the max-over-ranks of the timing."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, outdir):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import oracle
    import tina_inputs as ti
    from paper_2408_16551_b200 import shard
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    P, M, F = 16, 4, 37
    case = ti.pfb_case(P, M, F, seed=9)
    x = case.x[0]
    f_lo, f_hi, s_lo, s_hi = shard.shard_frames(x.shape[0], P, M, world, rank)
    part = oracle.pfb(x[s_lo:s_hi], P, M, case.window)
    assert part.shape[0] == f_hi - f_lo
    np.save(os.path.join(outdir, f"part{rank}.npy"), part)
    t = shard.max_over_ranks(1.0 + rank)
    assert t == float(world)
    streams = list(shard.shard_streams(5, world, rank))
    np.save(os.path.join(outdir, f"streams{rank}.npy"), np.array(streams))
    dist.barrier()
    dist.destroy_process_group()


def test_frame_shards_reproduce_full_result(tmp_path, oracle):
    import torch.multiprocessing as mp
    import tina_inputs as ti
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    P, M, F = 16, 4, 37
    case = ti.pfb_case(P, M, F, seed=9)
    full = oracle.pfb(case.x[0], P, M, case.window)
    got = np.concatenate([np.load(tmp_path / f"part{r}.npy") for r in range(world)])
    assert np.array_equal(got, full)
    s = np.concatenate([np.load(tmp_path / f"streams{r}.npy") for r in range(world)])
    assert s.tolist() == [0, 1, 2, 3, 4]


@pytest.mark.parametrize("n,P,M,world", [(4099 * 16, 16, 4, 3), (64, 16, 4, 4), (1 << 20, 4096, 8, 8)])
def test_shard_frames_cover_exactly(n, P, M, world):
    from paper_2408_16551_b200 import shard
    F = n // P - M + 1
    nxt = 0
    for r in range(world):
        f_lo, f_hi, s_lo, s_hi = shard.shard_frames(n, P, M, world, r)
        assert f_lo == nxt and f_hi >= f_lo
        nxt = f_hi
        if f_hi > f_lo:
            assert s_lo == f_lo * P and s_hi == (f_hi + M - 1) * P and s_hi <= n
            assert (s_hi - s_lo) // P - M + 1 == f_hi - f_lo
    assert nxt == F
