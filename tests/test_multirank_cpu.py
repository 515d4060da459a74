"""World-size-2 gloo test of the N > 1 path on CPU: coarse-channel sharding (no data-path collective),
max-over-ranks timing, and that the shards together reproduce the single-process batch result (oracle as checker)."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_2303_11557_b200 import shard, synth  # noqa: E402


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


N_COARSE, N_IN, N_FFT, T = 5, 6, 16, 4


def _worker(rank, world, port, out_dir):
    from oracle import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    mine = shard.coarse_channels_for_rank(N_COARSE, rank, world)
    res = {}
    for c in mine:
        spec = synth.GaussSpec(N_IN, N_FFT * T, N_FFT, sigma=16.0, rho=0.1, tones=[], seed=77, coarse=c)
        res[c] = oracle.fx(synth.gauss_voltages(spec), N_FFT, N_FFT, T, 1)
    # the slowest rank defines the step time
    t_max = shard.max_over_ranks(10.0 + rank)
    assert t_max == 10.0 + world - 1
    rate = shard.whole_job_rate(2.0, world, t_max)
    assert rate == pytest.approx(2.0 * world / t_max)
    # no data-path collective: each rank just writes its own channels
    np.savez(os.path.join(out_dir, f"rank{rank}.npz"), **{f"c{c}": v for c, v in res.items()})
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_shard_coarse_channels(tmp_path):
    from oracle import oracle
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    got = {}
    for r in range(world):
        with np.load(tmp_path / f"rank{r}.npz") as z:
            for k in z.files:
                assert k not in got, "a coarse channel was processed by two ranks"
                got[k] = z[k]
    assert sorted(got) == [f"c{c}" for c in range(N_COARSE)]
    for c in range(N_COARSE):
        spec = synth.GaussSpec(N_IN, N_FFT * T, N_FFT, sigma=16.0, rho=0.1, tones=[], seed=77, coarse=c)
        ref = oracle.fx(synth.gauss_voltages(spec), N_FFT, N_FFT, T, 1)
        assert np.array_equal(got[f"c{c}"], ref)


def test_assignment_is_a_partition():
    for world in (1, 2, 3, 8):
        for n in (0, 1, 7, 8, 24):
            seen = sorted(c for r in range(world) for c in shard.coarse_channels_for_rank(n, r, world))
            assert seen == list(range(n))
    with pytest.raises(ValueError):
        shard.coarse_channels_for_rank(4, 2, 2)


def test_max_over_ranks_without_group_is_identity():
    assert shard.max_over_ranks(3.5) == 3.5
