"""The N > 1 ("replicas only") host path on CPU: two gloo ranks, no GPU.  Each rank takes its own batch of seeded
candidate kernel sets, runs the ORACLE on a tiny workload in place of the CUDA library (the host logic under test is
the partition, the max-over-ranks timing and the global best), and the ranks must agree on the result."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2106_15350_b200 import replicas, synth


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import oracle as orc
        w = synth.scaled(synth.WORKLOADS["tiny_mnist"], 300, 100, 3)
        trx, try_, tex, tey = synth.make_dataset(w)
        ker = synth.make_kernels(w, w.n_cand, first=replicas.first_candidate(rank, w.n_cand))
        oa = orc.make_arch(w.in_h, w.in_w, w.in_c, w.layers)
        r = orc.search(oa, trx, try_, tex, tey, w.n_classes, w.C, ker, feature_scale=w.feature_scale)
        t_local = 1.0 + rank          # pretend rank 1 is slower
        t_max = replicas.max_over_ranks(t_local)
        acc, gidx = replicas.global_best(float(r["acc"][r["best"]]), int(r["best"]), rank, w.n_cand)
        q.put((rank, t_max, acc, gidx, ker.tobytes(), [float(a) for a in r["acc"]]))
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_partition_time_and_best():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=240) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (_, t0, a0, g0, k0, accs0), (_, t1, a1, g1, k1, accs1) = out
    assert t0 == t1 == 2.0                                   # the slowest rank's time, on every rank
    assert k0 != k1                                          # disjoint candidate batches
    w = synth.scaled(synth.WORKLOADS["tiny_mnist"], 300, 100, 3)
    both = synth.make_kernels(w, 2 * w.n_cand)               # the global stream = rank 0's batch then rank 1's
    assert both[: w.n_cand].tobytes() == k0 and both[w.n_cand:].tobytes() == k1
    allacc = accs0 + accs1
    assert (a0, g0) == (a1, g1)
    assert g0 == int(np.argmax(allacc)) and a0 == max(allacc)   # first maximum over the global stream
    assert replicas.job_throughput(world, w.n_cand, 5, t0) == pytest.approx(2 * 3 * 5 / 2.0)


def test_single_process_is_identity():
    assert replicas.max_over_ranks(3.5) == 3.5
    assert replicas.global_best(0.9, 2, 0, 8) == (0.9, 2)
    assert replicas.first_candidate(3, 64) == 192
