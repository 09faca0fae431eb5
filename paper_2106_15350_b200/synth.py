"""Seeded synthetic inputs for the LB-CNN kernel-selection loop (shared by oracle tests and the CUDA path).

This module holds NO arithmetic of the method (no convolution, pooling, ELM): it only draws
images, labels and binary (+-1) kernel sets, with the shapes of BASELINE.json ``configs`` and the
recipe of DESIGN.md section "Input recipe".  Both the CPU oracle (``oracle/``) and the CUDA library
consume the byte arrays produced here; neither imports the other.

Randomness is a counter-based splitmix64 (no dependence on a library's stream):
    u64(seed, i) = mix(seed + (i + 1) * 0x9E3779B97F4A7C15)
The paper draws "randomly generated binary kernels ... in each loop iteration" (PAPER.md:115,
section IV.A) -- here each tap is +-1 with probability 1/2, independently.
The datasets the paper measures on (MNIST, GTSRB, ORL, VGG-face: PAPER.md:104,147,159,172) are not
available; these generators reproduce only their shapes, class counts and split sizes.
"""
from __future__ import annotations

import dataclasses
from typing import Dict, List, Tuple

import numpy as np

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)

# layer tuple fields (mirrors lbcnn_layer_t in include/lbcnn.h; plain data, no arithmetic)
CONV_FULL, CONV_DEPTHWISE = 0, 1
ACT_NONE, ACT_RELU = 0, 1


def _mix(z: np.ndarray) -> np.ndarray:
    z = z.astype(np.uint64, copy=True)
    with np.errstate(over="ignore"):
        z ^= z >> np.uint64(30)
        z *= _M1
        z ^= z >> np.uint64(27)
        z *= _M2
        z ^= z >> np.uint64(31)
    return z


def splitmix64_scalar(x: int) -> int:
    """mix() of a single 64-bit integer (python ints)."""
    return int(_mix(np.array([x & 0xFFFFFFFFFFFFFFFF], dtype=np.uint64))[0])


class Stream:
    """Counter-based stream: the i-th draw depends only on (seed, tag, i)."""

    def __init__(self, seed: int, tag: int = 0):
        self.key = np.uint64(splitmix64_scalar((seed + 0x632BE59BD9B4E019 * (tag + 1)) & 0xFFFFFFFFFFFFFFFF))
        self.pos = 0

    def u64(self, n: int) -> np.ndarray:
        idx = np.arange(self.pos + 1, self.pos + n + 1, dtype=np.uint64)
        self.pos += n
        with np.errstate(over="ignore"):
            return _mix(self.key + idx * _GOLDEN)

    def uniform(self, n: int, lo: float = 0.0, hi: float = 1.0) -> np.ndarray:
        u = (self.u64(n) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)
        return lo + (hi - lo) * u

    def integers(self, n: int, m: int) -> np.ndarray:
        """uniform integers in [0, m)."""
        return np.minimum((self.uniform(n) * m).astype(np.int64), m - 1)

    def normal(self, n: int) -> np.ndarray:
        m = (n + 1) // 2
        u1 = 1.0 - self.uniform(m)  # (0,1]
        u2 = self.uniform(m)
        r = np.sqrt(-2.0 * np.log(u1))
        z = np.concatenate([r * np.cos(2 * np.pi * u2), r * np.sin(2 * np.pi * u2)])
        return z[:n]


# --------------------------------------------------------------------------------------------
# workload descriptions (BASELINE.json configs[0..4] = config 1..5; P6 = paper anchor, parity only)
# --------------------------------------------------------------------------------------------

@dataclasses.dataclass(frozen=True)
class Layer:
    conv_type: int
    n_kernels: int
    ksize: int
    act: int
    pool_k: int
    pool_s: int
    pool_p: int
    pool_cover_all: int


@dataclasses.dataclass(frozen=True)
class Workload:
    name: str
    config: int                 # 1..5, 6 = paper anchor
    in_h: int
    in_w: int
    in_c: int
    layers: Tuple[Layer, ...]
    n_train: int
    n_test: int
    n_classes: int
    n_cand: int
    C: float
    generator: str              # "blobs" | "lowrank" | "faces"
    zipf_s: float = 0.0
    feature_scale: float = 1.0 / 255.0


def _full(n, k, pk, ps, pp=0, cover=0):
    return Layer(CONV_FULL, n, k, ACT_NONE, pk, ps, pp, cover)


def _dw(m, k, pk, ps, pp=0, cover=0):
    return Layer(CONV_DEPTHWISE, m, k, ACT_NONE, pk, ps, pp, cover)


WORKLOADS: Dict[str, Workload] = {
    # configs[0]: tiny MNIST-shaped
    "tiny_mnist": Workload("tiny_mnist", 1, 28, 28, 1, (_full(4, 3, 4, 4),), 2000, 500, 10, 8, 1e3, "blobs"),
    # configs[1]: MNIST-shaped reduced-subset search (the configuration `metric` is quoted on)
    "mnist": Workload("mnist", 2, 28, 28, 1, (_full(10, 3, 2, 2), _full(20, 3, 2, 2)), 20000, 10000, 10, 64, 1e4, "blobs"),
    # configs[2]: GTSRB-shaped
    "gtsrb": Workload("gtsrb", 3, 32, 32, 3, (_full(16, 3, 2, 2), _full(32, 3, 2, 2)), 30000, 12630, 43, 128, 1e4, "lowrank", zipf_s=0.7),
    # configs[3]: ORL-shaped faces
    "orl": Workload("orl", 4, 112, 92, 1, (_full(8, 5, 4, 4),), 280, 120, 40, 1024, 1e2, "faces"),
    # configs[4]: VGG-face-shaped
    "vggface": Workload("vggface", 5, 64, 64, 3, (_full(16, 3, 2, 2), _full(32, 3, 2, 2)), 20000, 5000, 100, 32, 1e4, "lowrank"),
    # P6: the paper's own architecture family: depthwise (16,20), pool (4,2,1,cover_all)
    "paper_anchor": Workload("paper_anchor", 6, 28, 28, 1, (_dw(16, 3, 4, 2, 1, 1), _dw(20, 3, 4, 2, 1, 1)), 1000, 500, 10, 2, 1e4, "blobs"),
    # the same architecture at the size of the paper's Table I run ("first 20k" MNIST training samples,
    # F = 15680, primal 15680 x 15680 system): a measured context line (bench.py --workload paper_table1), not a BASELINE config
    "paper_table1": Workload("paper_table1", 6, 28, 28, 1, (_dw(16, 3, 4, 2, 1, 1), _dw(20, 3, 4, 2, 1, 1)), 20000, 10000, 10, 4, 1e4, "blobs"),
}


def scaled(w: Workload, n_train: int = None, n_test: int = None, n_cand: int = None) -> Workload:
    """Same workload at a reduced size (for parity tests the oracle finishes in seconds)."""
    return dataclasses.replace(
        w,
        n_train=w.n_train if n_train is None else n_train,
        n_test=w.n_test if n_test is None else n_test,
        n_cand=w.n_cand if n_cand is None else n_cand,
    )


def data_seed(config: int) -> int:
    return 21061535000 + config


def kernel_seed(config: int, k: int) -> int:
    return splitmix64_scalar(0x4C42434E00000000 + 4096 * config + k)


def layer_channels(w: Workload) -> List[Tuple[int, int]]:
    """(Cin, Cout) per layer: FULL -> n_kernels; DEPTHWISE -> Cin * multiplier."""
    out, c = [], w.in_c
    for L in w.layers:
        co = L.n_kernels if L.conv_type == CONV_FULL else c * L.n_kernels
        out.append((c, co))
        c = co
    return out


def kernel_set_size(w: Workload) -> Tuple[int, int]:
    """(#int8 weights, #int32 biases) per candidate; weights are [n_kernels][Cin][k][k] per layer."""
    nw = nb = 0
    for L, (ci, co) in zip(w.layers, layer_channels(w)):
        nw += L.n_kernels * ci * L.ksize * L.ksize
        nb += co
    return nw, nb


def make_kernels(w: Workload, n_cand: int = None, first: int = 0) -> np.ndarray:
    """int8 [n_cand][n_weights], every entry -1 or +1 (PAPER.md:88 `kers`)."""
    n_cand = w.n_cand if n_cand is None else n_cand
    nw, _ = kernel_set_size(w)
    out = np.empty((n_cand, nw), dtype=np.int8)
    for k in range(n_cand):
        bits = Stream(kernel_seed(w.config, first + k)).u64(nw) >> np.uint64(63)
        out[k] = (bits.astype(np.int8) << 1) - 1
    return out


# --------------------------------------------------------------------------------------------
# image generators
# --------------------------------------------------------------------------------------------

def _blob(hh, ww, cy, cx, sg):
    yy, xx = np.mgrid[0:hh, 0:ww]
    return np.exp(-((yy - cy) ** 2 + (xx - cx) ** 2) / (2.0 * sg * sg))


def _gen_blobs(w: Workload, n: int, seed: int):
    """MNIST-shaped: class-conditional Gaussian-blob templates + shift + gain + uniform noise."""
    pad = 3
    ch, cw = w.in_h + 2 * pad, w.in_w + 2 * pad
    st = Stream(seed, 0)
    base = np.zeros((ch, cw))
    for _ in range(2):
        cy, cx, sg = st.uniform(1, 9, ch - 9)[0], st.uniform(1, 9, cw - 9)[0], st.uniform(1, 3.0, 5.0)[0]
        base += 100.0 * _blob(ch, cw, cy, cx, sg)
    T = np.empty((w.n_classes, ch, cw))
    for c in range(w.n_classes):
        T[c] = base
        for _ in range(2):
            cy, cx, sg = st.uniform(1, 9, ch - 9)[0], st.uniform(1, 9, cw - 9)[0], st.uniform(1, 1.5, 3.5)[0]
            T[c] += 120.0 * _blob(ch, cw, cy, cx, sg)
    # one stream per per-sample variable, so that sample i does not depend on how many samples are drawn
    y = Stream(seed, 1).integers(n, w.n_classes).astype(np.int32)
    dy = Stream(seed, 4).integers(n, 2 * pad + 1)
    dx = Stream(seed, 5).integers(n, 2 * pad + 1)
    g = 1.0 + 0.3 * Stream(seed, 6).uniform(n, -1.0, 1.0)
    sn = Stream(seed, 2)
    X = np.empty((n, w.in_h, w.in_w, 1), dtype=np.uint8)
    chunk = 4096
    iy = np.arange(w.in_h)[None, :, None]
    ix = np.arange(w.in_w)[None, None, :]
    for a in range(0, n, chunk):
        b = min(n, a + chunk)
        m = b - a
        t = T[y[a:b, None, None], dy[a:b, None, None] + iy, dx[a:b, None, None] + ix]
        noise = sn.uniform(m * w.in_h * w.in_w, -60.0, 60.0).reshape(m, w.in_h, w.in_w)
        X[a:b, :, :, 0] = np.clip(np.rint(g[a:b, None, None] * t + noise), 0, 255).astype(np.uint8)
    return X, y


def _box(v: np.ndarray, k: int, axis: int) -> np.ndarray:
    """length-preserving moving average of width k along axis (zeros beyond the ends)."""
    p = k // 2
    padw = [(0, 0)] * v.ndim
    padw[axis] = (p, p)
    vp = np.pad(v, padw)
    cs = np.cumsum(vp, axis=axis)
    z = np.zeros_like(np.take(cs, [0], axis=axis))
    cs = np.concatenate([z, cs], axis=axis)
    n = v.shape[axis]
    hi = np.take(cs, np.arange(k, k + n), axis=axis)
    lo = np.take(cs, np.arange(0, n), axis=axis)
    return (hi - lo) / k


def _lowrank(st: Stream, m: int, hh: int, ww: int, cc: int, rank: int = 4) -> np.ndarray:
    """m fields of shape (hh, ww, cc): per channel sum_r u_r v_r^T with box-smoothed normal u, v."""
    u = _box(st.normal(m * cc * rank * hh).reshape(m, cc, rank, hh), 5, 3) * 2.2
    v = _box(st.normal(m * cc * rank * ww).reshape(m, cc, rank, ww), 5, 3) * 2.2
    f = np.einsum("mcrh,mcrw->mhwc", u, v)
    return f


def _labels_from_prior(st: Stream, n: int, n_classes: int, zipf_s: float) -> np.ndarray:
    p = (np.arange(n_classes) + 1.0) ** (-zipf_s) if zipf_s > 0 else np.ones(n_classes)
    cdf = np.cumsum(p / p.sum())
    return np.minimum(np.searchsorted(cdf, st.uniform(n), side="right"), n_classes - 1).astype(np.int32)


def _gen_lowrank(w: Workload, n: int, seed: int, class_amp: float, var_amp: float, noise: float):
    """GTSRB-/VGG-face-shaped RGB: shared field + per-class low-rank template + per-sample field + noise."""
    st = Stream(seed, 0)
    M = _lowrank(st, 1, w.in_h, w.in_w, w.in_c)[0]
    T = 40.0 * M[None] + class_amp * _lowrank(st, w.n_classes, w.in_h, w.in_w, w.in_c)
    y = _labels_from_prior(Stream(seed, 1), n, w.n_classes, w.zipf_s)
    g = 1.0 + 0.25 * Stream(seed, 4).uniform(n, -1.0, 1.0)
    sv = Stream(seed, 2)
    sn = Stream(seed, 3)
    X = np.empty((n, w.in_h, w.in_w, w.in_c), dtype=np.uint8)
    chunk = 1024
    for a in range(0, n, chunk):
        b = min(n, a + chunk)
        m = b - a
        var = _lowrank(sv, m, w.in_h, w.in_w, w.in_c)
        nz = sn.uniform(m * w.in_h * w.in_w * w.in_c, -noise, noise).reshape(m, w.in_h, w.in_w, w.in_c)
        img = 128.0 + g[a:b, None, None, None] * T[y[a:b]] + var_amp * var + nz
        X[a:b] = np.clip(np.rint(img), 0, 255).astype(np.uint8)
    return X, y


def _smooth_field(st: Stream, m: int, hh: int, ww: int) -> np.ndarray:
    f = st.normal(m * hh * ww).reshape(m, hh, ww)
    f = _box(_box(f, 9, 1), 9, 2)
    return f / f.std(axis=(1, 2), keepdims=True)


def _gen_faces(w: Workload, n_train: int, n_test: int, seed: int, id_amp: float, var_amp: float, noise: float):
    """ORL-shaped: per identity smooth random field; per_id images per identity, identity-major;
    the first 70 % of each identity's images go to train, the rest to test (7 + 3 at full size)."""
    assert n_train % w.n_classes == 0 and n_test % w.n_classes == 0
    ptr, pte = n_train // w.n_classes, n_test // w.n_classes
    per = ptr + pte
    st = Stream(seed, 0)
    M = _smooth_field(st, 1, w.in_h, w.in_w)[0]
    I = _smooth_field(st, w.n_classes, w.in_h, w.in_w)
    sv = Stream(seed, 2)
    sn = Stream(seed, 3)
    n = per * w.n_classes
    var = _smooth_field(sv, n, w.in_h, w.in_w)
    nz = sn.uniform(n * w.in_h * w.in_w, -noise, noise).reshape(n, w.in_h, w.in_w)
    ident = np.repeat(np.arange(w.n_classes), per)
    img = 128.0 + 60.0 * M[None] + id_amp * I[ident] + var_amp * var + nz
    X = np.clip(np.rint(img), 0, 255).astype(np.uint8)[..., None]
    j = np.tile(np.arange(per), w.n_classes)
    tr, te = j < ptr, j >= ptr
    y = ident.astype(np.int32)
    return X[tr], y[tr], X[te], y[te]


# amplitudes per workload, frozen after calibration with the oracle ("Input recipe"): the oracle's
# accuracies must stay below 100 % and spread by at least 2 percentage points across the candidates
AMPS: Dict[str, Dict[str, float]] = {
    "gtsrb": dict(class_amp=7.0, var_amp=22.0, noise=75.0),
    "vggface": dict(class_amp=4.0, var_amp=22.0, noise=75.0),
    "orl": dict(id_amp=13.0, var_amp=40.0, noise=25.0),
}


def make_dataset(w: Workload):
    """Returns (train_images u8 NHWC, train_labels i32, test_images u8 NHWC, test_labels i32).
    Train = first n_train samples of the stream, test = the next n_test ("first 20k")."""
    seed = data_seed(w.config if w.config != 6 else 2)   # P6 uses config-2 images
    if w.generator == "blobs":
        X, y = _gen_blobs(w, w.n_train + w.n_test, seed)
    elif w.generator == "lowrank":
        X, y = _gen_lowrank(w, w.n_train + w.n_test, seed, **AMPS[w.name])
    elif w.generator == "faces":
        return _gen_faces(w, w.n_train, w.n_test, seed, **AMPS[w.name])
    else:
        raise ValueError(w.generator)
    nt = w.n_train
    return (np.ascontiguousarray(X[:nt]), np.ascontiguousarray(y[:nt]),
            np.ascontiguousarray(X[nt:]), np.ascontiguousarray(y[nt:]))
