#!/usr/bin/env python
"""Writes tests/golden/fullsize_<workload>.npz: the ORACLE's result for whole candidates of BASELINE.json
configs[2] (gtsrb) and configs[4] (vggface) at FULL size (SURVEY.md 8(c) "cache oracle outputs ... keyed by
config + seeds so parity runs do not recompute them").

    python tests/golden/make_fullsize_golden.py [gtsrb] [vggface]

Calls only oracle/ and the seeded generators (paper_2106_15350_b200/synth.py holds no arithmetic of the
method); nothing here touches the CUDA path.  One candidate costs the oracle minutes (half Gram
N F^2 / 2 fp64 multiply-adds + F^3 / 6 for the Cholesky, plain loops), which is why the result is stored.

Stored per workload (candidate indices CANDS): W as float32 (its rounding, 6e-8, is far inside the 1e-3
tolerance), the predicted labels, the correct count, the top-1 / top-2 logit margin of every test sample
(to diagnose a disagreement as a near-tie) and `key` = CRC32s of the exact input bytes the oracle saw;
tests/test_gpu_parity.py recomputes the key from the generators and falls back to running the oracle
if it does not match.
"""
import os
import sys
import time
import zlib

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import oracle as orc                      # noqa: E402
from paper_2106_15350_b200 import synth               # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))
# first, middle and last candidate of the launch bench.py times (128 / 32 candidates); W is kept for candidate 0 only
# (8192 x 100 floats each: the others are compared through their labels and counts)
CANDS = {"gtsrb": [0, 64, 127], "vggface": [0, 16, 31]}
W_STORED = (0,)


def input_key(trx, try_, tex, tey, ker_k, C, scale) -> np.ndarray:
    parts = [trx, try_, tex, tey, ker_k, np.array([C, scale], dtype=np.float64)]
    return np.array([zlib.crc32(np.ascontiguousarray(p).tobytes()) for p in parts], dtype=np.int64)


def oracle_candidate(w, trx, try_, tex, tey, ker_k):
    """expand -> fit -> score of ONE candidate with the oracle; returns (W, pred, correct, margin, info)."""
    oa = orc.make_arch(w.in_h, w.in_w, w.in_c, w.layers)
    s = float(np.float32(w.feature_scale))
    Htr = orc.expand(oa, trx, ker_k).astype(np.float64) * s
    W, info, _ = orc.elm_fit(Htr, try_, w.n_classes, w.C)
    del Htr
    Hte = orc.expand(oa, tex, ker_k).astype(np.float64) * s
    pred, corr, margin = orc.elm_score(Hte, W, tey, want_margin=True)
    return W, pred, corr, margin, info


def path_of(name):
    return os.path.join(HERE, "fullsize_%s.npz" % name)


def main(names):
    orc.build()
    for name in names:
        w = synth.WORKLOADS[name]
        trx, try_, tex, tey = synth.make_dataset(w)
        ker = synth.make_kernels(w)
        out = {"cands": np.array(CANDS[name], dtype=np.int64)}
        old = dict(np.load(path_of(name))) if os.path.exists(path_of(name)) else {}
        for k in CANDS[name]:
            key = input_key(trx, try_, tex, tey, ker[k], w.C, float(np.float32(w.feature_scale)))
            if ("key_%d" % k) in old and np.array_equal(old["key_%d" % k], key):      # stored for these very input bytes: keep
                for f in ("W_%d", "pred_%d", "correct_%d", "margin_%d", "key_%d"):
                    if (f % k) in old:
                        out[f % k] = old[f % k]
                print("%s candidate %d: kept (input key matches)" % (name, k), flush=True)
                continue
            t0 = time.perf_counter()
            W, pred, corr, margin, info = oracle_candidate(w, trx, try_, tex, tey, ker[k])
            assert info == 0
            if k in W_STORED:
                out["W_%d" % k] = W.astype(np.float32)
            out["pred_%d" % k] = pred.astype(np.int16)
            out["correct_%d" % k] = np.array(corr, dtype=np.int64)
            out["margin_%d" % k] = margin.astype(np.float32)
            out["key_%d" % k] = input_key(trx, try_, tex, tey, ker[k], w.C, float(np.float32(w.feature_scale)))
            print("%s candidate %d: accuracy %.4f, %.1f s on %d threads" %
                  (name, k, corr / float(w.n_test), time.perf_counter() - t0, orc.n_threads()), flush=True)
        np.savez_compressed(path_of(name), **out)
        print("wrote", path_of(name), os.path.getsize(path_of(name)), "bytes", flush=True)


if __name__ == "__main__":
    main(sys.argv[1:] or ["gtsrb", "vggface"])
