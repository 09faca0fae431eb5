"""Seeded input generators: determinism, shapes, alphabet (no method arithmetic lives in synth.py)."""
import numpy as np

from paper_2106_15350_b200 import synth


def test_workload_table_matches_baseline_configs():
    W = synth.WORKLOADS
    assert (W["tiny_mnist"].n_train, W["tiny_mnist"].n_test, W["tiny_mnist"].n_cand, W["tiny_mnist"].C) == (2000, 500, 8, 1e3)
    assert (W["mnist"].n_train, W["mnist"].n_test, W["mnist"].n_cand, W["mnist"].C) == (20000, 10000, 64, 1e4)
    assert (W["gtsrb"].n_train, W["gtsrb"].n_test, W["gtsrb"].n_classes, W["gtsrb"].n_cand) == (30000, 12630, 43, 128)
    assert (W["orl"].n_train, W["orl"].n_test, W["orl"].n_classes, W["orl"].n_cand, W["orl"].C) == (280, 120, 40, 1024, 1e2)
    assert (W["vggface"].n_train, W["vggface"].n_test, W["vggface"].n_classes, W["vggface"].n_cand) == (20000, 5000, 100, 32)
    assert synth.kernel_set_size(W["mnist"]) == (10 * 9 + 20 * 10 * 9, 30)
    assert synth.kernel_set_size(W["paper_anchor"]) == (16 * 9 + 20 * 16 * 9, 16 + 320)


def test_kernels_are_pm1_and_counter_based():
    w = synth.WORKLOADS["mnist"]
    k = synth.make_kernels(w, 6)
    assert k.dtype == np.int8 and k.shape == (6, 1890) and set(np.unique(k)) == {-1, 1}
    assert abs(k.mean()) < 0.05
    assert np.array_equal(synth.make_kernels(w, 2, first=3), k[3:5])      # candidate k depends only on (config, k)


def test_datasets_deterministic_and_shaped():
    for name, (ntr, nte) in {"tiny_mnist": (64, 32), "gtsrb": (80, 40), "orl": (80, 40), "vggface": (100, 50)}.items():
        w = synth.scaled(synth.WORKLOADS[name], ntr, nte, 2)
        a = synth.make_dataset(w)
        b = synth.make_dataset(w)
        for x, y in zip(a, b):
            assert np.array_equal(x, y)
        trx, try_, tex, tey = a
        assert trx.dtype == np.uint8 and trx.shape == (ntr, w.in_h, w.in_w, w.in_c) and tex.shape[0] == nte
        assert try_.dtype == np.int32 and try_.min() >= 0 and try_.max() < w.n_classes
        assert trx.std() > 5


def test_train_prefix_property():
    # train = first n samples of the stream: a smaller workload is a prefix of a larger one (blobs / lowrank generators)
    w1 = synth.scaled(synth.WORKLOADS["tiny_mnist"], 50, 20, 1)
    w2 = synth.scaled(synth.WORKLOADS["tiny_mnist"], 70, 20, 1)
    a, b = synth.make_dataset(w1), synth.make_dataset(w2)
    assert np.array_equal(a[0], b[0][:50]) and np.array_equal(a[1], b[1][:50])
