"""lbcnn_evolve_candidates_static: the genetic generation step for callers that cannot supply a workspace.

Who they are (include/lbcnn.h has the long form): code that gets input and output buffers from its host application and has
no device allocator of its own, processes whose HBM is entirely owned by a start-up memory pool, and loops that must avoid
the device-wide stall of cudaMalloc / cudaFree.  For them the ranking scratch (8 bytes per candidate) is a fixed 128 KB array
inside liblbcnn.so instead of a slice of a caller-allocated workspace, which caps the population at 16384 candidates.

This file checks that the two entry points are interchangeable: same inputs -> byte-for-byte the same next generation (the
comparison every test of this byte-valued step uses, test_gpu_parity.py::test_genetic_generator_bit_exact_and_improves
included).  It runs two calls back to back, the second on a SMALLER population than the first, so a result that depended on
what the previous call left in the shared array would show up.  It is named to be collected last: it must pass both after the
whole suite has used the GPU and alone in a fresh process, where its first call is also the once-per-device address look-up.
"""
import numpy as np
import pytest
import torch

from paper_2106_15350_b200 import binding as lb

pytestmark = pytest.mark.gpu


def _population(rng, K, nw):
    ker = (rng.integers(0, 2, size=(K, nw)) * 2 - 1).astype(np.int8)
    acc = rng.integers(50, 60, size=K).astype(np.float32) / 100.0      # many exact ties: the ranking falls back on the index
    acc[K // 2] = -1.0                                                  # one failed fit, ranked last
    return torch.from_numpy(ker).cuda(), torch.from_numpy(acc).cuda()


def test_static_scratch_entry_equals_workspace_entry_twice_in_a_row():
    rng = np.random.default_rng(2106)
    with_ws = lb.Handle(0)       # the existing path: draws its scratch from a torch-allocated workspace
    no_ws = lb.Handle(0)         # never given a workspace: the static entry point must not need one
    try:
        # two consecutive calls; the second population is smaller, so stale entries of the first would lie beyond its clear
        for K, nw, elite, ppm, seed, gen in [(700, 513, 5, 20000, 7, 2), (24, 1890, 4, 5000, 123456789012345, 0)]:
            ker, acc = _population(rng, K, nw)
            got = no_ws.evolve_candidates_static(ker, acc, elite, ppm, seed, gen)
            ref = with_ws.evolve_candidates(ker, acc, elite, ppm, seed, gen)
            torch.cuda.synchronize()
            assert got.dtype == torch.int8 and got.shape == ref.shape
            assert torch.equal(got, ref), (K, nw)
            assert set(np.unique(got.cpu().numpy()).tolist()) <= {-1, 1}
        assert no_ws._ws is None
        # the same call repeated gives the same bytes (nothing of the previous call's scratch leaks into the next)
        again = no_ws.evolve_candidates_static(ker, acc, elite, ppm, seed, gen)
        torch.cuda.synchronize()
        assert torch.equal(again, ref)
    finally:
        with_ws.close()
        no_ws.close()


def test_static_scratch_entry_refuses_populations_beyond_its_array():
    h = lb.Handle(0)
    try:
        K = lb.EVOLVE_STATIC_MAX_CAND
        ker = torch.ones((K + 1, 3), dtype=torch.int8, device="cuda")
        acc = torch.zeros((K + 1,), dtype=torch.float32, device="cuda")
        with pytest.raises(lb.LbcnnError) as e:
            h.evolve_candidates_static(ker, acc, 1, 0, 1, 0)
        assert e.value.status == lb.ERR_STATIC_LIMIT
        assert "built-in scratch" in str(e.value)
        # exactly at the limit it runs, and agrees with the workspace path
        got = h.evolve_candidates_static(ker[:K], acc[:K], 2, 500000, 3, 1)
        ref = h.evolve_candidates(ker[:K], acc[:K], 2, 500000, 3, 1)
        torch.cuda.synchronize()
        assert torch.equal(got, ref)
    finally:
        h.close()
