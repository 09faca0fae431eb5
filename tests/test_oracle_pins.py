"""Pins for the CPU oracle (oracle/lbcnn_oracle.c) against things other than itself.

Every test here runs without a GPU.  What fixes the expected values:
  * digits printed in the paper (tests/golden/paper_shapes.txt, cited per row);
  * hand-worked examples (tests/golden/worked_examples.txt);
  * library routines computing the same textbook operation another way
    (torch.nn.functional.conv2d / max_pool2d in fp64, scipy.signal.correlate2d,
    numpy.linalg.solve / lstsq / pinv);
  * brute-force window enumeration in pure Python on tiny inputs;
  * closed forms and invariants (sign flip, linearity, primal == dual, C -> inf, scale identity ...).
"""
import math
import os

import numpy as np
import pytest
import scipy.signal
import torch
import torch.nn.functional as TF

from oracle import oracle as orc

GOLD = os.path.join(os.path.dirname(__file__), "golden")
FULL, DW = 0, 1
PAPER_POOL = (4, 2, 1, 1)  # max_pooling_2d(ksize=4, stride=2, pad=1, cover_all=True)


# ------------------------------------------------------------------------------------------------
# fixtures parsing
# ------------------------------------------------------------------------------------------------
def _paper_rows():
    rows = []
    for line in open(os.path.join(GOLD, "paper_shapes.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, shape, classes, mult, bits, F, cite = [t.strip() for t in line.split("|")]
        h, w, c = [int(t) for t in shape.split()]
        conv_s, elm_s = [t.strip() for t in bits.split(",")]
        rows.append(dict(name=name, h=h, w=w, c=c, classes=int(classes), mult=[int(t) for t in mult.split(",")],
                         conv=conv_s, elm=elm_s, F=F, cite=cite))
    return rows


def _worked():
    out, cur = {}, None
    for line in open(os.path.join(GOLD, "worked_examples.txt")):
        line = line.rstrip("\n")
        if line.startswith("#") or not line.strip():
            continue
        if line.startswith("["):
            cur = line.strip()[1:-1]
            out[cur] = {}
            continue
        key, val = line.split(":", 1)
        if key == "cite":
            continue
        out[cur][key.strip()] = np.array([[float(t) for t in r.split()] for r in val.split(";")])
    return out


WORKED = _worked()


def _printed_matches(value_bits: int, printed: str) -> bool:
    """the paper prints k-bits truncated to the digits shown"""
    d = len(printed.split(".")[1]) if "." in printed else 0
    kb = value_bits / 1000.0
    return math.floor(kb * 10 ** d + 1e-9) / 10 ** d == float(printed)


# ------------------------------------------------------------------------------------------------
# shape arithmetic
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,paper,p220,p440", [(28, 14, 14, 7), (14, 7, 7, 3), (7, 4, 3, 1), (32, 16, 16, 8),
                                               (16, 8, 8, 4), (64, 32, 32, 16), (112, 56, 56, 28), (92, 46, 46, 23)])
def test_pool_out_size_table(n, paper, p220, p440):
    # 28->14->7 is printed (28x28 -> F=15680 = 7*7*320); 7->4 follows from Table II (40,2,2)
    assert orc.pool_out_size(n, *PAPER_POOL) == paper
    assert orc.pool_out_size(n, 2, 2, 0, 0) == p220
    assert orc.pool_out_size(n, 4, 4, 0, 0) == p440


def test_pool_out_size_invalid():
    assert orc.pool_out_size(3, 4, 4, 0, 0) < 1          # window larger than the image
    assert orc.pool_out_size(0, 2, 2, 0, 0) < 1
    assert orc.pool_out_size(4, 2, 2, 2, 0) < 1          # first window lies entirely in the padding
    assert orc.pool_out_size(4, 1, 1, 0, 0) == 4         # (1,1,0,0) = no pooling


@pytest.mark.parametrize("row", _paper_rows(), ids=lambda r: r["name"])
def test_paper_printed_sizes(row):
    layers = [(DW, m, 3, 0) + PAPER_POOL for m in row["mult"]]
    arch = orc.make_arch(row["h"], row["w"], row["c"], layers)
    F, (ho, wo, co) = orc.feature_dim(arch)
    assert F == ho * wo * co
    assert co == row["c"] * int(np.prod(row["mult"]))
    conv_bits, elm_bits = orc.param_bits(arch, row["classes"])
    assert elm_bits == F * row["classes"] * 8
    if row["F"] != "-":
        assert F == int(row["F"]), row["cite"]
    if row["conv"] != "-":
        assert _printed_matches(conv_bits, row["conv"]), (conv_bits, row["cite"])
        assert _printed_matches(elm_bits, row["elm"]), (elm_bits, row["cite"])


def test_cover_all_is_pinned_by_table_II():
    # MNIST (40,2,2): 204.8 kbit = F*10*8 -> F = 2560 = 4*4*160, i.e. 7 -> 4 (cover_all); floor pooling would give 3*3*160
    arch = orc.make_arch(28, 28, 1, [(DW, 40, 3, 0) + PAPER_POOL, (DW, 2, 3, 0) + PAPER_POOL, (DW, 2, 3, 0) + PAPER_POOL])
    assert orc.feature_dim(arch)[0] == 2560
    arch_floor = orc.make_arch(28, 28, 1, [(DW, 40, 3, 0, 4, 2, 1, 0)] + [(DW, 2, 3, 0, 4, 2, 1, 0)] * 2)
    assert orc.feature_dim(arch_floor)[0] == 3 * 3 * 160


@pytest.mark.parametrize("name,shape,layers,F", [
    ("cfg1", (28, 28, 1), [(FULL, 4, 3, 0, 4, 4, 0, 0)], 196),
    ("cfg2", (28, 28, 1), [(FULL, 10, 3, 0, 2, 2, 0, 0), (FULL, 20, 3, 0, 2, 2, 0, 0)], 980),
    ("cfg3", (32, 32, 3), [(FULL, 16, 3, 0, 2, 2, 0, 0), (FULL, 32, 3, 0, 2, 2, 0, 0)], 2048),
    ("cfg4", (112, 92, 1), [(FULL, 8, 5, 0, 4, 4, 0, 0)], 5152),
    ("cfg5", (64, 64, 3), [(FULL, 16, 3, 0, 2, 2, 0, 0), (FULL, 32, 3, 0, 2, 2, 0, 0)], 8192),
])
def test_config_feature_dims(name, shape, layers, F):
    # BASELINE.json configs[0..4]: "4*7*7=196", "20*7*7=980", "32*8*8=2048", "8*28*23=5152", "32*16*16=8192"
    assert orc.feature_dim(orc.make_arch(*shape, layers))[0] == F


def test_invalid_arch_rejected():
    with pytest.raises(ValueError):
        orc.feature_dim(orc.make_arch(3, 3, 1, [(FULL, 2, 3, 0, 4, 4, 0, 0)]))
    with pytest.raises(ValueError):
        orc.feature_dim(orc.make_arch(8, 8, 1, [(FULL, 2, 4, 0, 2, 2, 0, 0)]))  # even kernel size


# ------------------------------------------------------------------------------------------------
# convolution
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("ex", ["conv4x4_checker", "conv4x4_ones"])
def test_conv_and_pool_worked_examples(ex):
    g = WORKED[ex]
    img = g["image"].astype(np.int64)[None, :, :, None]
    z = orc.conv(FULL, 1, 3, img, g["kernel"].astype(np.int8)[None, None])
    assert np.array_equal(z[0, :, :, 0], g["z"].astype(np.int64))
    for key, geom in (("pool_2_2_0_0", (2, 2, 0, 0)), ("pool_4_2_1_1", (4, 2, 1, 1)), ("pool_4_4_0_0", (4, 4, 0, 0))):
        u = orc.maxpool(z, *geom)
        assert np.array_equal(u[0, :, :, 0], g[key].astype(np.int64)), key


@pytest.mark.parametrize("k,ex", [(3, "tapcount3"), (5, "tapcount5")])
def test_conv_tap_counts(k, ex):
    img = np.ones((1, k, k, 1), dtype=np.int64)
    z = orc.conv(FULL, 1, k, img, np.ones((1, 1, k, k), dtype=np.int8))
    assert np.array_equal(z[0, :, :, 0], WORKED[ex]["z"].astype(np.int64))
    # FULL convolution over Cin all-ones channels multiplies the count by Cin
    img3 = np.ones((1, k, k, 3), dtype=np.int64)
    z3 = orc.conv(FULL, 2, k, img3, np.ones((2, 3, k, k), dtype=np.int8))
    assert np.array_equal(z3[0, :, :, 1], 3 * WORKED[ex]["z"].astype(np.int64))


def _rand_case(rng, n, h, w, cin, nk, k):
    a = rng.integers(-300, 300, size=(n, h, w, cin)).astype(np.int64)
    wt = (rng.integers(0, 2, size=(nk, cin, k, k)) * 2 - 1).astype(np.int8)
    b = rng.integers(-50, 50, size=(nk if True else 0,)).astype(np.int32)
    return a, wt, b


@pytest.mark.parametrize("k", [3, 5])
def test_conv_full_vs_library(k):
    """FULL conv == torch.conv2d (cross-correlation, zero pad) in fp64 == scipy correlate2d summed over channels."""
    rng = np.random.default_rng(100 + k)
    for _ in range(25):
        n, h, w = rng.integers(1, 3), rng.integers(1, 9), rng.integers(1, 9)
        cin, nk = rng.integers(1, 4), rng.integers(1, 5)
        a, wt, b = _rand_case(rng, n, h, w, cin, nk, k)
        z = orc.conv(FULL, nk, k, a, wt, b)
        ref = TF.conv2d(torch.from_numpy(a).double().permute(0, 3, 1, 2), torch.from_numpy(wt).double(),
                        bias=torch.from_numpy(b).double(), padding=(k - 1) // 2).permute(0, 2, 3, 1).numpy()
        assert np.array_equal(z, ref.astype(np.int64))
        o = int(rng.integers(0, nk))
        sc = sum(scipy.signal.correlate2d(a[0, :, :, c], wt[o, c].astype(np.int64), mode="same", boundary="fill")
                 for c in range(cin)) + b[o]
        assert np.array_equal(z[0, :, :, o], sc)


def test_conv_depthwise_vs_library_and_channel_order():
    """DEPTHWISE: out channel c*M+m uses w[m][c] on input channel c (reading R3).
    torch groups=Cin with weight[(c*M+m), 0] is the same operation."""
    rng = np.random.default_rng(7)
    for _ in range(25):
        n, h, w = 2, rng.integers(2, 8), rng.integers(2, 8)
        cin, M = rng.integers(1, 4), rng.integers(1, 4)
        a, wt, _ = _rand_case(rng, n, h, w, cin, M, 3)
        b = rng.integers(-9, 9, size=(cin * M,)).astype(np.int32)
        z = orc.conv(DW, M, 3, a, wt, b)
        wg = np.zeros((cin * M, 1, 3, 3))
        for c in range(cin):
            for m in range(M):
                wg[c * M + m, 0] = wt[m, c]
        ref = TF.conv2d(torch.from_numpy(a).double().permute(0, 3, 1, 2), torch.from_numpy(wg), bias=torch.from_numpy(b).double(),
                        padding=1, groups=int(cin)).permute(0, 2, 3, 1).numpy()
        assert np.array_equal(z, ref.astype(np.int64))


def test_conv_sign_flip_and_linearity():
    rng = np.random.default_rng(3)
    a, wt, _ = _rand_case(rng, 2, 6, 7, 3, 4, 3)
    a2 = rng.integers(0, 255, size=a.shape).astype(np.int64)
    z = orc.conv(FULL, 4, 3, a, wt)
    wf = wt.copy()
    wf[2] = -wf[2]
    zf = orc.conv(FULL, 4, 3, a, wf)
    assert np.array_equal(zf[..., 2], -z[..., 2])                       # flipping kernel 2 negates channel 2 ...
    assert np.array_equal(np.delete(zf, 2, axis=3), np.delete(z, 2, axis=3))   # ... and nothing else
    assert np.array_equal(orc.conv(FULL, 4, 3, a + a2, wt), z + orc.conv(FULL, 4, 3, a2, wt))


def test_conv_is_correlation_not_flipped():
    # a single 1 at the centre of a 3x3 image reproduces the kernel rotated by 180 degrees under correlation
    img = np.zeros((1, 3, 3, 1), dtype=np.int64)
    img[0, 1, 1, 0] = 1
    ker = np.array([[1, 1, -1], [1, -1, -1], [-1, 1, 1]], dtype=np.int8)
    z = orc.conv(FULL, 1, 3, img, ker[None, None])[0, :, :, 0]
    assert np.array_equal(z, ker[::-1, ::-1])


# ------------------------------------------------------------------------------------------------
# max-pool
# ------------------------------------------------------------------------------------------------
def _pool_brute(z, k, s, p, cover):
    n, h, w, c = z.shape
    def osz(m):
        span = m + 2 * p - k
        return (-(-span // s) if cover else span // s) + 1
    ho, wo = osz(h), osz(w)
    out = np.empty((n, ho, wo, c), dtype=np.int64)
    for b in range(n):
        for i in range(ho):
            for j in range(wo):
                for o in range(c):
                    cells = [z[b, y, x, o] for y in range(i * s - p, i * s - p + k) for x in range(j * s - p, j * s - p + k)
                             if 0 <= y < h and 0 <= x < w]
                    out[b, i, j, o] = max(cells)
    return out


@pytest.mark.parametrize("geom", [(2, 2, 0, 0), (4, 4, 0, 0), (4, 2, 1, 1), (3, 2, 1, 0), (3, 3, 0, 1), (1, 1, 0, 0)])
def test_maxpool_brute_force(geom):
    rng = np.random.default_rng(11)
    for _ in range(20):
        h, w = rng.integers(geom[0], 12), rng.integers(geom[0], 12)
        z = rng.integers(-1000, 1000, size=(2, h, w, 3)).astype(np.int64)
        assert np.array_equal(orc.maxpool(z, *geom), _pool_brute(z, *geom))


@pytest.mark.parametrize("geom,n", [((4, 2, 1, 1), 28), ((4, 2, 1, 1), 7), ((2, 2, 0, 0), 14), ((4, 4, 0, 0), 28)])
def test_maxpool_vs_torch(geom, n):
    k, s, p, cover = geom
    rng = np.random.default_rng(5)
    z = rng.integers(-500, 500, size=(2, n, n, 2)).astype(np.int64)
    ref = TF.max_pool2d(torch.from_numpy(z).double().permute(0, 3, 1, 2), k, s, p, ceil_mode=bool(cover)).permute(0, 2, 3, 1).numpy()
    assert np.array_equal(orc.maxpool(z, *geom), ref.astype(np.int64))


def test_maxpool_constant_and_negative():
    z = np.full((1, 7, 7, 2), -5, dtype=np.int64)
    u = orc.maxpool(z, *PAPER_POOL)
    assert u.shape == (1, 4, 4, 2) and np.all(u == -5)      # padding (-inf) never wins, even for negative inputs
    z = np.full((1, 8, 8, 1), 3, dtype=np.int64)
    assert np.all(orc.maxpool(z, 2, 2, 0, 0) == 3)


# ------------------------------------------------------------------------------------------------
# expander = composition + CHW flatten
# ------------------------------------------------------------------------------------------------
def _torch_expand(images, layers, kernels):
    x = torch.from_numpy(images.astype(np.float64)).permute(0, 3, 1, 2)
    off = 0
    for (ct, nk, k, act, pk, ps, pp, cov) in layers:
        cin = x.shape[1]
        nw = nk * cin * k * k
        wt = kernels[off:off + nw].reshape(nk, cin, k, k).astype(np.float64)
        off += nw
        if ct == FULL:
            x = TF.conv2d(x, torch.from_numpy(wt), padding=(k - 1) // 2)
        else:
            wg = np.zeros((cin * nk, 1, k, k))
            for c in range(cin):
                for m in range(nk):
                    wg[c * nk + m, 0] = wt[m, c]
            x = TF.conv2d(x, torch.from_numpy(wg), padding=(k - 1) // 2, groups=cin)
        if act == 1:
            x = torch.relu(x)
        x = TF.max_pool2d(x, pk, ps, pp, ceil_mode=bool(cov))
    return x.flatten(1).numpy().astype(np.int64)        # NCHW flatten = (o*Hout + i)*Wout + j  (reading R7)


@pytest.mark.parametrize("shape,layers", [
    ((28, 28, 1), [(FULL, 4, 3, 0, 4, 4, 0, 0)]),
    ((28, 28, 1), [(FULL, 10, 3, 0, 2, 2, 0, 0), (FULL, 20, 3, 0, 2, 2, 0, 0)]),
    ((16, 16, 3), [(FULL, 16, 3, 0, 2, 2, 0, 0), (FULL, 32, 3, 0, 2, 2, 0, 0)]),
    ((24, 20, 1), [(FULL, 8, 5, 0, 4, 4, 0, 0)]),
    ((28, 28, 1), [(DW, 16, 3, 0) + PAPER_POOL, (DW, 20, 3, 0) + PAPER_POOL]),
    ((14, 14, 2), [(DW, 3, 3, 1) + PAPER_POOL, (FULL, 5, 3, 1, 2, 2, 0, 0), (DW, 2, 3, 0) + PAPER_POOL]),
])
def test_expand_vs_torch_pipeline(shape, layers):
    rng = np.random.default_rng(42)
    h, w, c = shape
    images = rng.integers(0, 256, size=(3, h, w, c)).astype(np.uint8)
    arch = orc.make_arch(h, w, c, layers)
    nw, cc = 0, c
    for (ct, nk, k, *_r) in layers:
        nw += nk * cc * k * k
        cc = nk if ct == FULL else cc * nk
    kernels = (rng.integers(0, 2, size=nw) * 2 - 1).astype(np.int8)
    u = orc.expand(arch, images, kernels)
    assert np.array_equal(u, _torch_expand(images, layers, kernels))


def test_expand_bias_and_relu():
    rng = np.random.default_rng(8)
    images = rng.integers(0, 256, size=(2, 8, 8, 1)).astype(np.uint8)
    ker = (rng.integers(0, 2, size=3 * 9) * 2 - 1).astype(np.int8)
    arch = orc.make_arch(8, 8, 1, [(FULL, 3, 3, 0, 1, 1, 0, 0)])
    u0 = orc.expand(arch, images, ker)
    bias = np.array([5, -7, 100], dtype=np.int32)
    ub = orc.expand(arch, images, ker, bias)
    assert np.array_equal(ub.reshape(2, 3, 64), u0.reshape(2, 3, 64) + bias[None, :, None])   # CHW: channel-major blocks
    archr = orc.make_arch(8, 8, 1, [(FULL, 3, 3, 1, 1, 1, 0, 0)])
    assert np.array_equal(orc.expand(archr, images, ker), np.maximum(u0, 0))


def test_expand_integer_bounds_hold():
    # |z| <= 255 * taps for layer 1 (row E1 of the scope table): all-255 image, all-(+1) kernels reach it exactly
    images = np.full((1, 28, 28, 1), 255, dtype=np.uint8)
    arch = orc.make_arch(28, 28, 1, [(FULL, 4, 3, 0, 4, 4, 0, 0)])
    u = orc.expand(arch, images, np.ones(36, dtype=np.int8))
    assert u.max() == 2295


# ------------------------------------------------------------------------------------------------
# ELM fit
# ------------------------------------------------------------------------------------------------
def test_elm_worked_examples():
    g = WORKED["elm_3x2"]
    H = np.array([[1, 0], [0, 1], [1, 1]], dtype=np.float64)
    y = np.array([0, 1, 0], dtype=np.int32)
    for br in (1, 2):
        W, info, b = orc.elm_fit(H, y, 2, 1.0, force_branch=br)
        assert info == 0 and b == br
        assert np.allclose(W, g["W"], atol=1e-14)
    pred, corr, mar = orc.elm_score(H, g["W"], y, want_margin=True)
    assert list(pred) == [int(v) for v in g["pred"][0]] and corr == 3
    assert np.allclose(mar, [0.75, 0.25, 0.5])
    W, info, _ = orc.elm_fit(np.array([[1.0]]), np.array([0], dtype=np.int32), 2, 1.0)
    assert np.allclose(W, WORKED["elm_scalar"]["W"])


def test_elm_branch_rule():
    # listing: `if n_inputs < Ntr` -> 'LLL' (primal) else 'MMM' (dual); equality -> dual
    rng = np.random.default_rng(0)
    for n, F, want in ((10, 4, 1), (4, 10, 2), (6, 6, 2)):
        H = rng.normal(size=(n, F))
        y = rng.integers(0, 3, size=n).astype(np.int32)
        assert orc.elm_fit(H, y, 3, 10.0)[2] == want


def _onehot(y, c):
    T = np.zeros((len(y), c))
    T[np.arange(len(y)), y] = 1.0
    return T


def test_elm_primal_dual_and_dense_solve():
    """200 random instances, dims in [3,40]: primal == dual (push-through identity) and both equal
    numpy.linalg.solve on the normal equations; residual within 1e-6 * ||B|| (north_star)."""
    rng = np.random.default_rng(2024)
    for _ in range(200):
        n, F, c = rng.integers(3, 41), rng.integers(3, 41), rng.integers(2, 6)
        H = rng.normal(size=(n, F))
        y = rng.integers(0, c, size=n).astype(np.int32)
        Creg = float(10 ** rng.uniform(-1, 3))
        Wp, ip, _ = orc.elm_fit(H, y, c, Creg, force_branch=1)
        Wd, idd, _ = orc.elm_fit(H, y, c, Creg, force_branch=2)
        assert ip == 0 and idd == 0
        T = _onehot(y, c)
        A = H.T @ H + np.eye(F) / Creg
        B = H.T @ T
        ref = np.linalg.solve(A, B)
        nr = np.linalg.norm(ref)
        assert np.linalg.norm(Wp - Wd) <= 1e-6 * nr
        assert np.linalg.norm(Wp - ref) <= 1e-8 * nr
        assert np.linalg.norm(Wd - ref) <= 1e-8 * nr
        assert np.linalg.norm(A @ Wp - B) <= 1e-6 * np.linalg.norm(B)


def test_elm_large_C_is_least_squares():
    rng = np.random.default_rng(9)
    H = rng.normal(size=(60, 12))        # tall, full rank
    y = rng.integers(0, 4, size=60).astype(np.int32)
    T = _onehot(y, 4)
    W, info, _ = orc.elm_fit(H, y, 4, 1e12)
    assert info == 0
    assert np.allclose(W, np.linalg.lstsq(H, T, rcond=None)[0], atol=1e-8)
    assert np.allclose(W, np.linalg.pinv(H) @ T, atol=1e-8)


def test_elm_orthogonal_closed_form():
    # H^T H = alpha^2 I  ->  W = H^T T / (alpha^2 + 1/C)
    rng = np.random.default_rng(1)
    Q, _ = np.linalg.qr(rng.normal(size=(30, 8)))
    alpha, Creg = 3.0, 7.0
    H = alpha * Q
    y = rng.integers(0, 3, size=30).astype(np.int32)
    W, _, _ = orc.elm_fit(H, y, 3, Creg)
    assert np.allclose(W, H.T @ _onehot(y, 3) / (alpha ** 2 + 1 / Creg), atol=1e-12)


def test_elm_invariants():
    rng = np.random.default_rng(77)
    H = rng.normal(size=(50, 9))
    y = rng.integers(0, 4, size=50).astype(np.int32)
    Creg, s = 20.0, 1 / 255.0
    W, _, _ = orc.elm_fit(H, y, 4, Creg)
    # scale identity W(sH, C) = W(H, C s^2) / s  (reading R6)
    Ws, _, _ = orc.elm_fit(s * H, y, 4, Creg)
    W2, _, _ = orc.elm_fit(H, y, 4, Creg * s * s)
    assert np.allclose(Ws, W2 / s, rtol=1e-9, atol=1e-9)
    # label permutation permutes the columns of W
    perm = np.array([2, 0, 3, 1])
    Wp, _, _ = orc.elm_fit(H, perm[y].astype(np.int32), 4, Creg)
    assert np.allclose(Wp[:, perm], W, atol=1e-12)
    # columns of T sum to one: sum_c W[:,c] = A^-1 H^T 1
    A = H.T @ H + np.eye(9) / Creg
    assert np.allclose(W.sum(axis=1), np.linalg.solve(A, H.sum(axis=0)), atol=1e-10)
    # feature permutation leaves the logits unchanged
    fp = rng.permutation(9)
    Wf, _, _ = orc.elm_fit(H[:, fp], y, 4, Creg)
    assert np.allclose(H[:, fp] @ Wf, H @ W, atol=1e-10)


def test_elm_bad_arguments():
    H = np.ones((3, 2))
    with pytest.raises(ValueError):
        orc.elm_fit(H, np.array([0, 1, 5], dtype=np.int32), 2, 1.0)     # label out of range
    with pytest.raises(ValueError):
        orc.elm_fit(H, np.array([0, 1, 0], dtype=np.int32), 2, 0.0)     # C must be > 0


def test_elm_failure_return_is_first_bad_pivot():
    """Cholesky without jitter (R11): the return value is (index of the first pivot that is not > 0) + 1,
    LAPACK's convention.  Pinned by construction: a NaN in feature f poisons row / column f of H^T H only, so pivots
    0..f-1 are untouched and pivot f is the first to fail (primal); in the dual the same holds for the sample index."""
    rng = np.random.default_rng(5)
    y = rng.integers(0, 3, size=40).astype(np.int32)
    for f_bad, n_bad in ((2, 3), (0, 0), (7, 39)):
        H = rng.standard_normal((40, 8))
        H[n_bad, f_bad] = np.nan
        W, info, br = orc.elm_fit(H, y, 3, 1.0)
        assert br == 1 and info == f_bad + 1
        W, info, br = orc.elm_fit(H, y, 3, 1.0, force_branch=2)
        assert br == 2 and info == n_bad + 1
    # an indefinite system the ridge cannot repair: none exists for C > 0 with finite H (H^T H + I/C is SPD), and indeed
    # every finite instance factors
    for _ in range(20):
        H = rng.standard_normal((6, 9)) * 1e-8
        assert orc.elm_fit(H, np.arange(6, dtype=np.int32) % 3, 3, 1e12)[1] == 0


# ------------------------------------------------------------------------------------------------
# score
# ------------------------------------------------------------------------------------------------
def test_score_ties_and_accuracy():
    H = np.eye(4)
    W = np.array([[1.0, 1.0, 0.0], [0.0, 2.0, 2.0], [0.0, 0.0, 0.0], [-1.0, -3.0, -1.0]])
    pred, corr, _ = orc.elm_score(H, W, np.array([0, 1, 0, 1], dtype=np.int32))
    assert list(pred) == [0, 1, 0, 0]        # ties -> lowest index; all-zero row -> class 0
    assert corr == 3                         # 3 of 4 -> 0.75
    pred, corr, _ = orc.elm_score(H, W)
    assert corr is None


def test_score_matches_numpy_argmax():
    rng = np.random.default_rng(4)
    H, W = rng.normal(size=(200, 30)), rng.normal(size=(30, 7))
    y = rng.integers(0, 7, size=200).astype(np.int32)
    pred, corr, mar = orc.elm_score(H, W, y, want_margin=True)
    L = H @ W
    assert np.array_equal(pred, L.argmax(axis=1))
    assert corr == int((L.argmax(axis=1) == y).sum())
    srt = np.sort(L, axis=1)
    assert np.allclose(mar, srt[:, -1] - srt[:, -2])


# ------------------------------------------------------------------------------------------------
# search loop
# ------------------------------------------------------------------------------------------------
def test_search_best_worst_and_replay():
    from paper_2106_15350_b200 import synth
    w = synth.scaled(synth.WORKLOADS["tiny_mnist"], 300, 150, 5)
    trx, try_, tex, tey = synth.make_dataset(w)
    arch = orc.make_arch(w.in_h, w.in_w, w.in_c, w.layers)
    ker = synth.make_kernels(w)
    r = orc.search(arch, trx, try_, tex, tey, w.n_classes, w.C, ker, w.feature_scale, keep=True)
    assert r["best"] == int(np.argmax(r["acc"])) and r["worst"] == int(np.argmin(r["acc"]))
    assert np.all(r["acc"] == r["correct"] / 150.0)
    # replay of the best kernels alone reproduces the best accuracy exactly (PAPER.md:94 use_stored)
    r1 = orc.search(arch, trx, try_, tex, tey, w.n_classes, w.C, ker[r["best"]:r["best"] + 1], w.feature_scale)
    assert r1["best"] == 0 and r1["worst"] == 0 and r1["acc"][0] == r["acc"][r["best"]]
    # constant images, two classes: every kernel set gives identical rows -> prediction is one class for all
    cx = np.full((20, 28, 28, 1), 100, dtype=np.uint8)
    cy = np.zeros(20, dtype=np.int32)
    r2 = orc.search(arch, cx, cy, cx, cy, 2, 10.0, ker[:2], w.feature_scale)
    assert np.all(r2["acc"] == 1.0)


def test_search_failed_fit_is_excluded(monkeypatch):
    """a candidate whose fit fails gets accuracy -1 and info = pivot + 1, takes part in neither best nor worst
    (R13), and the other candidates' results are what a search over them alone gives."""
    from paper_2106_15350_b200 import synth
    w = synth.scaled(synth.WORKLOADS["tiny_mnist"], 250, 100, 4)
    trx, try_, tex, tey = synth.make_dataset(w)
    arch = orc.make_arch(w.in_h, w.in_w, w.in_c, w.layers)
    ker = synth.make_kernels(w)
    real_fit = orc.elm_fit
    calls = []

    def poisoned_fit(H, labels, n_classes, Creg, force_branch=0):
        calls.append(1)
        if len(calls) == 2:                    # the second candidate's features carry a NaN in feature 5
            H = H.copy()
            H[7, 5] = np.nan
        return real_fit(H, labels, n_classes, Creg, force_branch)

    monkeypatch.setattr(orc, "elm_fit", poisoned_fit)
    r = orc.search(arch, trx, try_, tex, tey, w.n_classes, w.C, ker, w.feature_scale, keep=True)
    monkeypatch.setattr(orc, "elm_fit", real_fit)
    assert r["info"].tolist() == [0, 6, 0, 0] and r["acc"][1] == -1.0 and r["W"][1] is None
    others = orc.search(arch, trx, try_, tex, tey, w.n_classes, w.C, ker[[0, 2, 3]], w.feature_scale)
    assert np.array_equal(r["acc"][[0, 2, 3]], others["acc"])
    assert r["best"] == [0, 2, 3][others["best"]] and r["worst"] == [0, 2, 3][others["worst"]]
    assert r["best"] != 1 and r["worst"] != 1


# ------------------------------------------------------------------------------------------------
# <= 8-bit output layer (R16)
# ------------------------------------------------------------------------------------------------
def test_quantize_worked_example_and_bounds():
    W = np.array([[0.5, -1.0], [0.25, 0.126]], dtype=np.float32)
    q, scale = orc.quantize_output_layer(W, 8)
    # 0.5 * 127 = 63.5 -> 64 (half to even), -127, 31.75 -> 32, 16.002 -> 16
    assert q.tolist() == [[64, -127], [32, 16]] and q.dtype == np.int8
    assert scale == np.float32(1.0 / 127.0)
    q2, s2 = orc.quantize_output_layer(W, 2)            # qmax = 1: sign of everything above half the maximum
    assert q2.tolist() == [[0, -1], [0, 0]] and s2 == np.float32(1.0)      # 0.5 -> rint(0.5) = 0 (half to even)
    rng = np.random.default_rng(3)
    for bits in (3, 5, 8):
        Wr = (rng.standard_normal((40, 7)) * rng.uniform(1e-3, 10)).astype(np.float32)
        q, scale = orc.quantize_output_layer(Wr, bits)
        qmax = 2 ** (bits - 1) - 1
        assert np.abs(q).max() == qmax                                     # the largest weight maps to +-qmax
        assert np.all(np.abs(Wr.astype(np.float64) - float(scale) * q) <= 0.5 * float(scale) * (1 + 1e-6))
        qa, sa = orc.quantize_output_layer(Wr * np.float32(4.0), bits)     # a power-of-two rescaling changes only the scale
        assert np.array_equal(qa, q) and sa == np.float32(4.0) * scale
        qd, _ = orc.quantize_output_layer((float(scale) * q).astype(np.float32), bits)      # a grid point stays put
        assert np.array_equal(qd, q)
    qz, sz = orc.quantize_output_layer(np.zeros((3, 2), dtype=np.float32), 8)
    assert not qz.any() and sz == 0.0
    with pytest.raises(ValueError):
        orc.quantize_output_layer(W, 9)


def test_score_q_is_exact_integer_arithmetic():
    rng = np.random.default_rng(9)
    U = rng.integers(-900000, 900000, size=(30, 17))
    q = rng.integers(-127, 128, size=(17, 5)).astype(np.int8)
    q[:, 4] = q[:, 1]                                                      # exact ties: the lower index must win
    y = rng.integers(0, 5, size=30).astype(np.int32)
    pred, corr, logits = orc.elm_score_q(U, q, y)
    for i in range(30):                                                    # python integers: no rounding anywhere
        row = [sum(int(U[i, f]) * int(q[f, c]) for f in range(17)) for c in range(5)]
        assert row == logits[i].tolist()
        assert pred[i] == row.index(max(row))
    assert (pred != 4).all() and corr == int((pred == y).sum())


# ------------------------------------------------------------------------------------------------
# genetic candidate generator (R17)
# ------------------------------------------------------------------------------------------------
def test_ga_generator_known_answers():
    # splitmix64 (Steele, Lea, Flood 2014) from state 0: the published first outputs are mix(1 * golden), mix(2 * golden)
    assert orc.ga_mix64(0x9E3779B97F4A7C15) == 0xE220A8397B1DCDAF
    assert orc.ga_mix64(2 * 0x9E3779B97F4A7C15) == 0x6E789E6AA1B965F4
    assert orc.ga_draw(1, 0, 0, 0) != orc.ga_draw(1, 0, 0, 1) != orc.ga_draw(1, 1, 0, 0)


def test_ga_generation_properties():
    rng = np.random.default_rng(21)
    K, nw = 24, 300
    ker = (rng.integers(0, 2, size=(K, nw)) * 2 - 1).astype(np.int8)
    acc = rng.uniform(0.5, 0.9, size=K).astype(np.float32)
    acc[5] = acc[11] = 0.95                   # a tie for the best: index 5 ranks first
    acc[3] = -1.0                             # a failed fit ranks last
    nxt, par, order = orc.evolve_candidates(ker, acc, n_elite=4, mut_ppm=0, seed=7, generation=2)
    assert order[0] == 5 and order[1] == 11 and order[-1] == 3
    assert list(order) == sorted(range(K), key=lambda i: (-acc[i], i))
    for j in range(4):                        # elitism: the best four, unchanged, in rank order
        assert np.array_equal(nxt[j], ker[order[j]]) and (par[j] == -1).all()
    assert set(np.unique(nxt)) <= {-1, 1}
    frac1 = []
    for j in range(4, K):                     # without mutation every tap comes from one of the two parents
        p1, p2 = par[j]
        assert np.all((nxt[j] == ker[p1]) | (nxt[j] == ker[p2]))
        differ = ker[p1] != ker[p2]
        if differ.sum() > 50:
            frac1.append((nxt[j][differ] == ker[p1][differ]).mean())
    assert 0.4 < np.mean(frac1) < 0.6         # uniform crossover
    # tournament: a parent is the better-ranked of its two draws, so parents rank better than uniform on average
    rank = np.empty(K, dtype=int); rank[order] = np.arange(K)
    assert rank[par[4:].ravel()].mean() < (K - 1) / 2.0
    # mutation only: with rate 1 every tap of the crossover result is flipped; with rate 2 % about 2 % are
    flipped, _, _ = orc.evolve_candidates(ker, acc, 4, 1000000, 7, 2)
    assert np.array_equal(flipped[4:], -nxt[4:]) and np.array_equal(flipped[:4], nxt[:4])
    some, _, _ = orc.evolve_candidates(ker, acc, 4, 20000, 7, 2)
    rate = (some[4:] != nxt[4:]).mean()
    assert 0.012 < rate < 0.028
    # counter-based: same arguments -> same children; another generation or seed -> different ones
    again, _, _ = orc.evolve_candidates(ker, acc, 4, 20000, 7, 2)
    assert np.array_equal(again, some)
    assert not np.array_equal(orc.evolve_candidates(ker, acc, 4, 20000, 7, 3)[0], some)
    assert not np.array_equal(orc.evolve_candidates(ker, acc, 4, 20000, 8, 2)[0], some)


def test_ga_nan_accuracy_ranks_last():
    """DESIGN.md R17: an accuracy that is not a number (0 / 0 when a caller scores on an empty test set, or garbage passed in)
    is ranked as minus infinity -- after the -1 of a failed fit, ties by index -- so order[] stays a permutation and the
    elites are real candidates."""
    rng = np.random.default_rng(5)
    K, nw = 12, 40
    ker = (rng.integers(0, 2, size=(K, nw)) * 2 - 1).astype(np.int8)
    acc = np.linspace(0.9, 0.5, K).astype(np.float32)
    acc[2] = np.nan; acc[7] = np.nan; acc[4] = -1.0
    nxt, par, order = orc.evolve_candidates(ker, acc, n_elite=K, mut_ppm=0, seed=1, generation=0)
    assert sorted(order.tolist()) == list(range(K))
    assert order.tolist() == [0, 1, 3, 5, 6, 8, 9, 10, 11, 4, 2, 7]
    assert np.array_equal(nxt, ker[order])


# ------------------------------------------------------------------------------------------------
# gradient refinement of the output layer (R18 = SPEC.md:324, 355)
# ------------------------------------------------------------------------------------------------
def test_refine_identity_order_and_first_step():
    rng = np.random.default_rng(2)
    H = rng.normal(size=(37, 6)); y = rng.integers(0, 3, size=37); W0 = rng.normal(size=(6, 3)) * 0.1
    W, losses = orc.refine_output_layer(H, y, W0, epochs=0, batch=8, lr=1e-3)
    assert np.array_equal(W, W0) and len(losses) == 0                      # epochs = 0 -> unchanged
    for n in (1, 2, 37, 20000, 30000):                                     # every epoch visits every sample exactly once
        a, b = orc.refine_order(5, 3, n)
        assert sorted(((a * np.arange(n, dtype=np.int64) + b) % n).tolist()) == list(range(n))
    # the first Adam step moves every weight by lr * sign(gradient) (m_hat / sqrt(v_hat) = g / |g|), whatever the data
    W1, _ = orc.refine_output_layer(H, y, W0, epochs=1, batch=37, lr=1e-2, eps=0.0)
    Z = H @ W0; P = np.exp(Z - Z.max(1, keepdims=True)); P /= P.sum(1, keepdims=True)
    P[np.arange(37), y] -= 1.0
    G = H.T @ P / 37.0
    assert np.allclose(W1, W0 - 1e-2 * np.sign(G), atol=1e-12)


def test_refine_adam_second_step_worked_example():
    """The recursion past its first step (m, v, BOTH bias corrections with t = 2, the running step counter), against the
    hand-worked values of tests/golden/worked_examples.txt [adam_two_steps] (R18 = SPEC.md:324, 355).  The same
    two steps are reached three ways: two epochs of one batch (the counter must run on across epochs), one epoch of two
    batches over the data written twice (it must run on inside an epoch; with n = 4 and an odd multiplier every batch of two
    consecutive draws holds one sample of each kind, whatever the seed), and a single step for the intermediate w1."""
    g = {k: v.ravel() for k, v in WORKED["adam_two_steps"].items()}
    sym = lambda x: np.array([[x, -x], [-x, x]])
    H = np.eye(2); y = np.array([0, 1]); W0 = np.zeros((2, 2))
    kw = dict(lr=0.1, beta1=0.9, beta2=0.999, eps=1e-8)
    W1, l1 = orc.refine_output_layer(H, y, W0, epochs=1, batch=2, **kw)
    assert np.allclose(W1, sym(g["w1"][0]), rtol=0, atol=1e-15) and abs(l1[0] - g["loss"][0]) < 1e-15
    for seed in (0, 1, 2, 3):
        W2, l2 = orc.refine_output_layer(H, y, W0, epochs=2, batch=2, seed=seed, **kw)
        assert np.allclose(W2, sym(g["w2"][0]), rtol=0, atol=2e-15), W2
        assert np.allclose(l2, g["loss"], rtol=0, atol=2e-15)
        H4 = np.vstack([H, H]); y4 = np.r_[y, y]
        W2b, l2b = orc.refine_output_layer(H4, y4, W0, epochs=1, batch=2, seed=seed, **kw)
        assert np.allclose(W2b, sym(g["w2"][0]), rtol=0, atol=2e-15), W2b
        assert abs(l2b[0] - g["loss"].mean()) < 2e-15
    # the golden block is consistent with itself (guards against a typo in the file, not against the oracle)
    assert abs(g["m2"][0] - (0.9 * g["m1"][0] + 0.1 * g["q"][0])) < 1e-17
    assert abs(g["mhat2"][0] - g["m2"][0] / g["c1"][0]) < 1e-16 and abs(g["vhat2"][0] - g["v2"][0] / g["c2"][0]) < 1e-16
    assert abs(g["w2"][0] - g["w1"][0] - 0.1 * g["mhat2"][0] / (math.sqrt(g["vhat2"][0]) + 1e-8)) < 1e-16
    # the two plausible mistakes named in the golden file land far away
    assert abs(g["w2"][0] - 0.2338324893844486) > 0.03


def test_refine_gradient_is_the_cross_entropy_gradient():
    # finite differences of the mean softmax cross-entropy against the step direction of one full batch
    rng = np.random.default_rng(8)
    for _ in range(5):
        n, F, c = 11, 4, 3
        H = rng.normal(size=(n, F)); y = rng.integers(0, c, size=n); W0 = rng.normal(size=(F, c)) * 0.3

        def loss(W):
            Z = 0.5 * (H @ W); Z = Z - Z.max(1, keepdims=True)
            return float(-(Z[np.arange(n), y] - np.log(np.exp(Z).sum(1))).mean())
        G = np.zeros_like(W0)
        for i in range(F):
            for j in range(c):
                d = np.zeros_like(W0); d[i, j] = 1e-6
                G[i, j] = (loss(W0 + d) - loss(W0 - d)) / 2e-6
        # one step with beta1 = beta2 = 0 and a huge eps turns Adam into W - lr * g / eps: read g back
        W1, l0 = orc.refine_output_layer(H, y, W0, 1, n, lr=1.0, beta1=0.0, beta2=0.0, eps=1e6, h_scale=0.5)
        g = (W0 - W1) * (1e6 + np.abs((W0 - W1) * 1e6))                    # g / (|g| + eps) = step  =>  g ~ step * eps (|g| << eps)
        assert np.allclose(g, G, rtol=1e-4, atol=1e-8)
        assert abs(l0[0] - loss(W0)) < 1e-12


def test_refine_descends_and_separates():
    rng = np.random.default_rng(4)
    n = 120
    y = rng.integers(0, 2, size=n)
    H = np.c_[np.where(y == 0, 1.0, -1.0) + 0.1 * rng.normal(size=n), rng.normal(size=n), np.ones(n)]
    W, losses = orc.refine_output_layer(H, y, np.zeros((3, 2)), epochs=30, batch=16, lr=5e-2, seed=1)
    assert losses[1] <= losses[0] and losses[2] <= losses[1] and losses[-1] < 0.2 * losses[0]
    pred, corr, _ = orc.elm_score(H, W, y.astype(np.int32))
    assert corr == n                                                        # separable toy set -> training accuracy 1
    W2, l2 = orc.refine_output_layer(H, y, np.zeros((3, 2)), epochs=30, batch=16, lr=5e-2, seed=1)
    assert np.array_equal(W, W2)                                            # deterministic given the seed
