"""world_size-2 gloo test (CPU) of the N>1 host logic bench.py uses: disjoint
per-rank beams, max-over-ranks timing, whole-job aggregation."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1112_0065_b200 import replicas
import workloads as W


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = W.CONFIGS["htru_gulp"].scaled(nchans=4, nsamps_out=256)
    beams = replicas.beam_indices(rank, 2)
    hashes = [W.sha256(W.generate(w, 10, beam=b)) for b in beams]
    dist.barrier()
    slow = replicas.max_over_ranks(1.0 + rank)          # rank 1 is the slow one
    q.put((rank, beams, hashes, slow, replicas.job_throughput(1000, world, slow)))
    dist.destroy_process_group()


def test_two_rank_replicas_gloo():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, b0, h0, s0, v0), (r1, b1, h1, s1, v1) = res
    assert b0 == [0, 1] and b1 == [2, 3]
    assert len(set(h0 + h1)) == 4                       # four distinct seeded beams
    assert s0 == s1 == 2.0                              # max over ranks on both
    assert v0 == v1 == 1000.0                           # 2 ranks * 1000 units / 2.0 s


def test_single_process_identity():
    assert replicas.max_over_ranks(3.5) == 3.5
    assert replicas.beam_indices(3, 13)[0] == 39


def _coincidence_worker(rank, world, port, q):
    """One beam subset per rank: local counts (here from the oracle -- no GPU in this test; on the GPU box they
    come from dedisp_rfi_beam_counts, tests/test_gpu_rfi_mask.py) -> all-reduce -> threshold."""
    from oracle import rfi_mask as RM
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    rng = np.random.default_rng(21)                       # the same 13 beams on every rank; rank r owns a slice
    x = rng.standard_normal((13, 1, 4096)).astype(np.float32)
    x[:, 0, 1000:1010] += 5.0                             # an all-beam burst (RFI) and a single-beam one (a pulse)
    x[3, 0, 2000:2005] += 8.0
    mean, sigma = np.zeros((13, 1), np.float32), np.ones((13, 1), np.float32)
    lo, hi = (0, 7) if rank == 0 else (7, 13)
    counts = torch.from_numpy(RM.beam_count(x[lo:hi], mean[lo:hi], sigma[lo:hi], 3.0).astype(np.uint8))
    replicas.allreduce_beam_counts(counts, 13)
    mask = (counts.numpy() >= 4).astype(np.uint8)
    want = RM.coincidence_mask(x, mean, sigma, 3.0, 4)
    q.put((rank, bool(np.array_equal(mask, want)), int(mask[0, 1000:1010].sum()), int(mask[0, 2000:2005].sum())))
    dist.destroy_process_group()


def test_two_rank_coincidence_counts_allreduce_gloo():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_coincidence_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, same, burst, pulse in res:
        assert same and burst == 10 and pulse == 0        # the all-beam burst is masked, the one-beam pulse is not


def test_allreduce_beam_counts_checks_its_arguments():
    c = torch.zeros((1, 8), dtype=torch.uint8)
    assert replicas.allreduce_beam_counts(c, 13) is c         # not distributed: identity
    with pytest.raises(ValueError):
        replicas.allreduce_beam_counts(c, 256)
    with pytest.raises(TypeError):
        replicas.allreduce_beam_counts(c.to(torch.int32), 13)
