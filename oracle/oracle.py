"""ctypes wrapper around oracle/lbcnn_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this.  It never imports the CUDA package.  The search loop below follows PAPER.md:88,94 (section
III, Cells 5/6): for every candidate kernel set, expand train and test sets, fit ELM0 on the train
features, score the test set, keep best and lowest.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lbcnn_oracle.c")
_LIB = os.path.join(_HERE, "liblbcnn_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp; rebuilt when the source is newer than the library."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-mavx2", "-ffp-contract=off", "-fPIC", "-shared", "-std=c11",
               "-Wall", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _Layer(C.Structure):
    _fields_ = [(n, C.c_int32) for n in
                ("conv_type", "n_kernels", "ksize", "act", "pool_k", "pool_s", "pool_p", "pool_cover_all")]


class _Arch(C.Structure):
    _fields_ = [("in_h", C.c_int32), ("in_w", C.c_int32), ("in_c", C.c_int32), ("n_layers", C.c_int32),
                ("layer", _Layer * 3)]


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.orc_pool_out_size.restype = C.c_int
        for f in ("orc_feature_dim", "orc_param_bits", "orc_conv", "orc_maxpool", "orc_expand", "orc_elm_fit",
                  "orc_elm_score"):
            getattr(_lib, f).restype = C.c_int
    return _lib


def n_threads() -> int:
    """threads the OpenMP runtime will use (OMP_NUM_THREADS or the cores visible to this process)."""
    v = os.environ.get("OMP_NUM_THREADS")
    if v:
        return int(v.split(",")[0])
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def make_arch(in_h: int, in_w: int, in_c: int, layers: Sequence) -> _Arch:
    """layers: objects/tuples with (conv_type, n_kernels, ksize, act, pool_k, pool_s, pool_p, pool_cover_all)."""
    a = _Arch()
    a.in_h, a.in_w, a.in_c, a.n_layers = in_h, in_w, in_c, len(layers)
    for i, L in enumerate(layers):
        t = tuple(L) if isinstance(L, (tuple, list)) else (
            L.conv_type, L.n_kernels, L.ksize, L.act, L.pool_k, L.pool_s, L.pool_p, L.pool_cover_all)
        for name, v in zip([f[0] for f in _Layer._fields_], t):
            setattr(a.layer[i], name, int(v))
    return a


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def pool_out_size(n, k, s, p, cover_all) -> int:
    return _load().orc_pool_out_size(int(n), int(k), int(s), int(p), int(cover_all))


def feature_dim(arch: _Arch) -> Tuple[int, Tuple[int, int, int]]:
    F = C.c_int64()
    hwc = (C.c_int32 * 3)()
    rc = _load().orc_feature_dim(C.byref(arch), C.byref(F), hwc)
    if rc:
        raise ValueError("invalid architecture (status %d)" % rc)
    return F.value, tuple(hwc)


def param_bits(arch: _Arch, n_classes: int) -> Tuple[int, int]:
    cb, eb = C.c_int64(), C.c_int64()
    rc = _load().orc_param_bits(C.byref(arch), int(n_classes), C.byref(cb), C.byref(eb))
    if rc:
        raise ValueError("invalid architecture (status %d)" % rc)
    return cb.value, eb.value


def conv(conv_type, n_kernels, ksize, a: np.ndarray, w: np.ndarray, bias: Optional[np.ndarray] = None) -> np.ndarray:
    """a: int64 [n][h][w][cin]; w: int8 [n_kernels][cin][k][k]; returns int64 [n][h][w][cout]."""
    a = np.ascontiguousarray(a, dtype=np.int64)
    w = np.ascontiguousarray(w, dtype=np.int8)
    n, h, ww, cin = a.shape
    cout = n_kernels if conv_type == 0 else cin * n_kernels
    assert w.size == n_kernels * cin * ksize * ksize
    b = None if bias is None else np.ascontiguousarray(bias, dtype=np.int32)
    z = np.empty((n, h, ww, cout), dtype=np.int64)
    rc = _load().orc_conv(int(conv_type), int(n_kernels), int(ksize), _p(a), C.c_int64(n), h, ww, cin, _p(w), _p(b), _p(z))
    if rc:
        raise ValueError("orc_conv status %d" % rc)
    return z


def maxpool(z: np.ndarray, k, s, p, cover_all) -> np.ndarray:
    z = np.ascontiguousarray(z, dtype=np.int64)
    n, h, w, c = z.shape
    ho, wo = pool_out_size(h, k, s, p, cover_all), pool_out_size(w, k, s, p, cover_all)
    if ho < 1 or wo < 1:
        raise ValueError("invalid pooling geometry")
    u = np.empty((n, ho, wo, c), dtype=np.int64)
    rc = _load().orc_maxpool(_p(z), C.c_int64(n), h, w, c, int(k), int(s), int(p), int(cover_all), _p(u))
    if rc:
        raise ValueError("orc_maxpool status %d" % rc)
    return u


def expand(arch: _Arch, images: np.ndarray, kernels: np.ndarray, bias: Optional[np.ndarray] = None) -> np.ndarray:
    """images u8 [n][H][W][C]; kernels int8 [n_weights] of ONE candidate; returns int64 [n][F] (exact integers)."""
    images = np.ascontiguousarray(images, dtype=np.uint8)
    kernels = np.ascontiguousarray(kernels, dtype=np.int8)
    assert images.shape[1:] == (arch.in_h, arch.in_w, arch.in_c), images.shape
    F, _ = feature_dim(arch)
    b = None if bias is None else np.ascontiguousarray(bias, dtype=np.int32)
    u = np.empty((images.shape[0], F), dtype=np.int64)
    rc = _load().orc_expand(C.byref(arch), _p(images), C.c_int64(images.shape[0]), _p(kernels), _p(b), _p(u))
    if rc:
        raise ValueError("orc_expand status %d" % rc)
    return u


def elm_fit(H: np.ndarray, labels: np.ndarray, n_classes: int, Creg: float, force_branch: int = 0):
    """H fp64 [n][F]; returns (W fp64 [F][classes], info, branch) -- branch 1 primal ('LLL'), 2 dual ('MMM')."""
    H = np.ascontiguousarray(H, dtype=np.float64)
    labels = np.ascontiguousarray(labels, dtype=np.int32)
    n, F = H.shape
    W = np.zeros((F, n_classes), dtype=np.float64)
    br = C.c_int32()
    info = _load().orc_elm_fit(_p(H), C.c_int64(n), C.c_int64(F), _p(labels), int(n_classes), C.c_double(Creg),
                               int(force_branch), _p(W), C.byref(br))
    if info < 0:
        raise ValueError("orc_elm_fit bad argument (%d)" % info)
    return W, info, br.value


def elm_score(H: np.ndarray, W: np.ndarray, labels: Optional[np.ndarray] = None, want_margin: bool = False):
    """returns (pred int32 [n], correct or None, margin or None)."""
    H = np.ascontiguousarray(H, dtype=np.float64)
    W = np.ascontiguousarray(W, dtype=np.float64)
    n, F = H.shape
    assert W.shape[0] == F
    classes = W.shape[1]
    lab = None if labels is None else np.ascontiguousarray(labels, dtype=np.int32)
    pred = np.empty(n, dtype=np.int32)
    corr = C.c_int64(0)
    mar = np.empty(n, dtype=np.float64) if want_margin else None
    rc = _load().orc_elm_score(_p(H), C.c_int64(n), C.c_int64(F), _p(W), classes, _p(lab), _p(pred), C.byref(corr), _p(mar))
    if rc:
        raise ValueError("orc_elm_score status %d" % rc)
    return pred, (corr.value if labels is not None else None), mar


def search(arch: _Arch, train_x, train_y, test_x, test_y, n_classes: int, Creg: float, kernels: np.ndarray,
           feature_scale: float = 1.0 / 255.0, bias: Optional[np.ndarray] = None, keep: bool = False):
    """The paper's trial loop: one trial per candidate kernel set.
    feature_scale is the fp32 number the library receives, widened to double (R6).
    Returns dict(acc [K] float64, correct [K], info [K], best, worst, W_best, and per-candidate W/pred if keep)."""
    K = kernels.shape[0]
    s = float(np.float32(feature_scale))
    acc = np.zeros(K)
    correct = np.zeros(K, dtype=np.int64)
    info = np.zeros(K, dtype=np.int32)
    Ws, preds = [], []
    for k in range(K):
        b = None if bias is None else bias[k]
        Htr = expand(arch, train_x, kernels[k], b).astype(np.float64) * s
        Hte = expand(arch, test_x, kernels[k], b).astype(np.float64) * s
        W, inf, _ = elm_fit(Htr, train_y, n_classes, Creg)
        info[k] = inf
        if inf:
            acc[k], correct[k] = -1.0, 0
            Ws.append(None); preds.append(None)
            continue
        pred, corr, _ = elm_score(Hte, W, test_y)
        correct[k] = corr
        acc[k] = corr / float(len(test_y))
        Ws.append(W); preds.append(pred)
    # first index of the maximum / of the minimum; failed fits (acc = -1) take part in neither (R13:
    # "lowest candidate index; failed fits are excluded").  All failed: 0 / 0.
    okk = np.nonzero(info == 0)[0]
    best = int(okk[np.argmax(acc[okk])]) if len(okk) else 0
    worst = int(okk[np.argmin(acc[okk])]) if len(okk) else 0
    out = dict(acc=acc, correct=correct, info=info, best=best, worst=worst, W_best=Ws[best])   # None if every fit failed
    if keep:
        out["W"], out["pred"] = Ws, preds
    return out


# ---- <= 8-bit fixed-point output layer ------------------------------------------------------------------
def quantize_output_layer(W: np.ndarray, bits: int = 8):
    """"weights represented as 8 bits integers" (Cell 12 "quantization with fixed-point ... maximum 8 bits",
    PAPER.md:94, 98).  The paper does not state the scheme; reading DESIGN.md R16: ONE symmetric scale per output layer,
        q = clip(rint(W * (qmax / max|W|)), -qmax, qmax),   qmax = 2^(bits-1) - 1,
    W taken as the fp32 numbers the fit returned, the product formed in fp64, rint = round half to even.
    Returns (q int8 [F][classes], scale float32 = max|W| / qmax), so that W ~ scale * q."""
    if not 2 <= bits <= 8:
        raise ValueError("bits must be 2..8")
    W32 = np.ascontiguousarray(W, dtype=np.float32)
    qmax = 2 ** (bits - 1) - 1
    m = float(np.max(np.abs(W32)))
    sf = (float(qmax) / m) if m > 0.0 else 0.0
    q = np.rint(W32.astype(np.float64) * sf)
    q = np.clip(q, -qmax, qmax).astype(np.int8)
    return q, np.float32(m / float(qmax))


def elm_score_q(U: np.ndarray, q: np.ndarray, labels: Optional[np.ndarray] = None):
    """Predict with the quantised layer on the INTEGER features U [n][F]: logits = U q in exact integer
    arithmetic, class = first index of the maximum (R12); the common positive scale cannot change the argmax.
    Returns (pred int32 [n], correct or None, logits int64 [n][classes])."""
    U = np.ascontiguousarray(U, dtype=np.int64)
    q = np.ascontiguousarray(q, dtype=np.int64)
    logits = U @ q
    pred = np.argmax(logits, axis=1).astype(np.int32)          # numpy returns the first maximum
    corr = None if labels is None else int((pred == np.asarray(labels)).sum())
    return pred, corr, logits


# ---- non-random candidate generator: one generation of a genetic search --------------------------------
# "nature inspired optimization methods (such as genetic algorithms or swarm intelligence methods)" are named as the way to
# go beyond random kernels; the paper gives no algorithm, so this is reading DESIGN.md R17, followed
# step by step.  The random numbers are a counter-based generator both sides implement: a splitmix64 finaliser keyed by
# (seed, generation, child, draw index).
_U64 = (1 << 64) - 1
_G1, _G2, _G3 = 0x9E3779B97F4A7C15, 0xBF58476D1CE4E5B9, 0x94D049BB133111EB


def ga_mix64(z: int) -> int:
    z &= _U64
    z = ((z ^ (z >> 30)) * _G2) & _U64
    z = ((z ^ (z >> 27)) * _G3) & _U64
    return z ^ (z >> 31)


def ga_draw(seed: int, generation: int, child: int, i: int) -> int:
    key = ga_mix64((seed & _U64) ^ ((_G1 * (generation + 1)) & _U64))
    ckey = ga_mix64(key + _G2 * (child + 1))
    return ga_mix64(ckey + _G1 * (i + 1))


def evolve_candidates(kernels: np.ndarray, acc: np.ndarray, n_elite: int, mut_ppm: int, seed: int, generation: int):
    """kernels int8 [K][n_weights] (+-1), acc [K] (the search's accuracies; a failed fit has -1).
    R17: 1. rank the candidates by accuracy, best first, equal accuracies by index (NaN counts as minus infinity);
         2. children 0 .. n_elite-1 are the n_elite best, unchanged, in rank order (elitism);
         3. every other child j draws two parents, each the better-ranked of two uniformly drawn candidates (binary
            tournament: draws 0,1 and 2,3, candidate = draw mod K), takes each tap from parent 1 or 2 by bit 0 of draw 4 + t
            (uniform crossover), and flips it when (draw >> 20) mod 10^6 < mut_ppm (mutation).
    Returns (next int8 [K][n_weights], parents int32 [K][2] with -1 for elites, order int32 [K])."""
    kernels = np.ascontiguousarray(kernels, dtype=np.int8)
    K, nw = kernels.shape
    a = np.asarray(acc, dtype=np.float32)
    a = np.where(np.isnan(a), np.float32(-np.inf), a)          # R17: not-a-number ranks as minus infinity (after failed fits)
    order = sorted(range(K), key=lambda i: (-float(a[i]), i))
    rank = [0] * K
    for r, i in enumerate(order):
        rank[i] = r
    nxt = np.empty_like(kernels)
    parents = np.full((K, 2), -1, dtype=np.int32)
    for j in range(K):
        if j < n_elite:
            nxt[j] = kernels[order[j]]
            continue
        c = [ga_draw(seed, generation, j, i) % K for i in range(4)]
        p1 = c[0] if rank[c[0]] <= rank[c[1]] else c[1]
        p2 = c[2] if rank[c[2]] <= rank[c[3]] else c[3]
        parents[j] = (p1, p2)
        for t in range(nw):
            d = ga_draw(seed, generation, j, 4 + t)
            v = int(kernels[p1, t]) if (d & 1) == 0 else int(kernels[p2, t])
            if ((d >> 20) % 1000000) < mut_ppm:
                v = -v
            nxt[j, t] = v
    return nxt, parents, np.array(order, dtype=np.int32)


# ---- gradient refinement of the output layer on the full set -----------------------------------------
# Cell 10 of the notebook trains "the output layer with the full dataset" with "the traditional Keras approach based on
# 'optimizers'" (+0.73 pp on MNIST) and names neither loss, optimiser nor schedule.  Reading
# DESIGN.md R18 = SPEC.md:324, 355: softmax cross-entropy, adaptive moment estimation (0.9, 0.999, 1e-8), mini-batches.
# The sample order of an epoch is the affine map i = (a j + b) mod N, gcd(a, N) = 1, with a and b from the counter-based
# generator above (both sides compute it on the host; no library shuffle).
def refine_order(seed: int, epoch: int, n: int):
    """(a, b) of epoch `epoch`: sample j of the epoch is (a j + b) mod n."""
    from math import gcd
    if n == 1:
        return 1, 0
    a = 1 + ga_draw(seed, epoch, 0, 0) % (n - 1)
    while gcd(a, n) != 1:
        a = a % (n - 1) + 1
    return a, ga_draw(seed, epoch, 0, 1) % n


def refine_output_layer(H: np.ndarray, labels: np.ndarray, W0: np.ndarray, epochs: int, batch: int, lr: float,
                        beta1: float = 0.9, beta2: float = 0.999, eps: float = 1e-8, seed: int = 0, h_scale: float = 1.0):
    """H [n][F] (stored features; logical feature = h_scale * H), W0 [F][classes] (e.g. the ELM fit).  fp64 throughout.
    Per mini-batch: Z = h_scale H_b W; P = softmax(Z) (row maximum subtracted); loss = -sum log P[i, y_i];
    G = h_scale H_b^T (P - T) / |batch|; Adam step on W.  Returns (W, mean loss per epoch)."""
    H = np.ascontiguousarray(H, dtype=np.float64)
    y = np.asarray(labels, dtype=np.int64)
    n, F = H.shape
    W = np.array(W0, dtype=np.float64, copy=True)
    c = W.shape[1]
    m = np.zeros_like(W); v = np.zeros_like(W)
    t = 0
    losses = []
    hs = float(np.float32(h_scale))
    for e in range(epochs):
        a, b = refine_order(seed, e, n)
        tot = 0.0
        for s0 in range(0, n, batch):
            j = np.arange(s0, min(n, s0 + batch), dtype=np.int64)
            idx = (a * j + b) % n
            Hb = H[idx]
            Z = hs * (Hb @ W)
            Z -= Z.max(axis=1, keepdims=True)
            E = np.exp(Z)
            P = E / E.sum(axis=1, keepdims=True)
            tot += float(-np.log(P[np.arange(len(idx)), y[idx]]).sum())
            D = P
            D[np.arange(len(idx)), y[idx]] -= 1.0
            G = hs * (Hb.T @ D) / float(len(idx))
            t += 1
            m = beta1 * m + (1.0 - beta1) * G
            v = beta2 * v + (1.0 - beta2) * G * G
            W -= lr * (m / (1.0 - beta1 ** t)) / (np.sqrt(v / (1.0 - beta2 ** t)) + eps)
        losses.append(tot / n)
    return W, np.array(losses)
