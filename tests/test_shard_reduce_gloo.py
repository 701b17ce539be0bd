"""World-size-2 check (gloo, CPU) of the multi-GPU reduction that bench.py --gpus N uses:
every rank digests the work items b with b % nranks == rank, the partial J~, K~ are summed with one all-reduce, and the
result equals the single-rank result.  The arithmetic here is the oracle's list digest (no GPU on this box); what is
tested is the dealing rule, its coverage (each item exactly once) and the collective plumbing."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

from paper_2407_09700_b200 import workloads as W  # noqa: E402


def shard_items(n_items: int, rank: int, nranks: int):
    """Same rule as the kernels: grid = ceil(n/nranks) blocks, block x handles item x*nranks + rank if it exists."""
    grid = (n_items + nranks - 1) // nranks
    return [x * nranks + rank for x in range(grid) if x * nranks + rank < n_items]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    basis, D, q = W.cfg1_class((1, 1, 1, 0), 2, nquartets=40, pool=6)
    mine = shard_items(len(q), rank, world)
    Jt, Kt = oracle.digest_list(basis, D, q[mine])
    J, K = torch.from_numpy(Jt), torch.from_numpy(Kt)
    dist.all_reduce(J); dist.all_reduce(K)
    cover = torch.zeros(len(q), dtype=torch.int64)
    cover[mine] = 1
    dist.all_reduce(cover)
    if rank == 0:
        Jf, Kf = oracle.digest_list(basis, D, q)
        out["dj"] = float(np.abs(J.numpy() - Jf).max() / np.abs(Jf).max())
        out["dk"] = float(np.abs(K.numpy() - Kf).max() / np.abs(Kf).max())
        out["cover"] = cover.tolist()
    dist.destroy_process_group()


def test_two_rank_partial_sums_equal_the_whole():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
        assert out["dj"] < 1e-13 and out["dk"] < 1e-13
        assert set(out["cover"]) == {1}


def test_dealing_rule_covers_every_block_once():
    for n in (0, 1, 5, 148, 1001):
        for nr in (1, 2, 3, 8):
            seen = sorted(sum((shard_items(n, r, nr) for r in range(nr)), []))
            assert seen == list(range(n))
