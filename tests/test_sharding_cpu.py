"""N > 1 host logic on CPU: world_size 2 over gloo -- beam assignment, distinct per-rank inputs, max-over-ranks timing
and summed candidate counts (the only exchanges of the sharded path)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    import sys
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    from paper_2606_27262_b200 import shard, synth
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        nbeam = 2
        beams = shard.beams_of_rank(rank, world, nbeam)
        w = synth.workload(4, nsamp=2048, nbeam=nbeam * world)
        sums = [int(synth.checksum(synth.generate(w, beam=b))) for b in beams]
        t = shard.max_over_ranks(10.0 + rank)            # "device time" of this rank
        c = shard.sum_over_ranks(100 * (rank + 1))
        np.save(os.path.join(out_dir, f"r{rank}.npy"), np.array([t, c] + beams + sums, dtype=np.float64))
        # the candidate merge: rank r brings 3 + 2r records of its local beams 0 and 1 (rank 1 more than rank 0)
        dt = np.dtype([("beam", "<i4"), ("trial", "<i4"), ("t", "<i4"), ("width", "<i4"), ("snr", "<f4")])
        loc = np.zeros(3 + 2 * rank, dtype=dt)
        loc["beam"] = np.arange(loc.size) % nbeam
        loc["trial"] = 10 * rank + np.arange(loc.size)
        loc["snr"] = 7.5 + rank
        merged = shard.merge_candidates(loc, rank, world, nbeam)
        assert (merged is None) == (rank != 0)
        if rank == 0:
            np.save(os.path.join(out_dir, "merged.npy"), merged)
        empty = shard.merge_candidates(loc[:0], rank, world, nbeam)       # nobody has anything
        assert empty is None or empty.size == 0
    finally:
        dist.destroy_process_group()


def test_two_ranks_share_nothing_but_scalars(tmp_path, synth):
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    r0, r1 = (np.load(tmp_path / f"r{r}.npy") for r in range(world))
    assert r0[0] == r1[0] == 11.0                       # max over ranks
    assert r0[1] == r1[1] == 300                        # summed candidate counts
    assert list(r0[2:4]) == [0, 1] and list(r1[2:4]) == [2, 3]          # disjoint beams, all covered
    assert len({*r0[4:6], *r1[4:6]}) == 4               # every beam has its own bytes
    m = np.load(tmp_path / "merged.npy")
    assert m.size == 3 + 5
    assert m["beam"].tolist() == [0, 1, 0, 2, 3, 2, 3, 2]               # local beams renumbered: rank 1 owns beams 2, 3
    assert m["trial"].tolist() == [0, 1, 2, 10, 11, 12, 13, 14] and m["snr"].tolist() == [7.5] * 3 + [8.5] * 5


def test_beam_assignment_covers_all_beams_once():
    from paper_2606_27262_b200 import shard
    for world in (1, 2, 4, 8):
        for nbeam in (1, 3, 64):
            got = sorted(b for r in range(world) for b in shard.beams_of_rank(r, world, nbeam))
            assert got == list(range(world * nbeam))
    with pytest.raises(ValueError):
        shard.beams_of_rank(2, 2, 1)
    assert shard.max_over_ranks(3.5) == 3.5 and shard.sum_over_ranks(7) == 7     # no process group: identity
