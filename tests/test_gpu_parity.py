"""Parity of the CUDA path (through the C ABI) with the CPU oracle on the same seeded inputs.

Tolerances are BASELINE.json `north_star`'s:
  integer features (feature_scale = 1)   bit-exact
  scaled features                        max relative error <= 1e-5 (exact zeros must match)
  ELM weights                            relative Frobenius error <= 1e-3
  predicted labels                       agreement >= 99.9 %
  accuracy                               within 0.2 percentage points
"""
import dataclasses
import zlib

import numpy as np
import pytest
import torch

from oracle import oracle as orc
from paper_2106_15350_b200 import binding as lb
from paper_2106_15350_b200 import synth

pytestmark = pytest.mark.gpu

TOL_FEAT_REL = 1e-5
TOL_W_FRO = 1e-3
TOL_LABEL_AGREE = 0.999
TOL_ACC_PP = 0.2


@pytest.fixture(scope="module")
def handle():
    h = lb.Handle(0)
    yield h
    h.close()


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _orc_arch(w):
    return orc.make_arch(w.in_h, w.in_w, w.in_c, w.layers)


def _small(name, n_train, n_test, n_cand):
    return synth.scaled(synth.WORKLOADS[name], n_train, n_test, n_cand)


# sizes chosen ragged on purpose (not multiples of 64 / of the CTA's candidate group of 8)
EXPAND_CASES = [("tiny_mnist", 37, 11), ("mnist", 21, 9), ("gtsrb", 13, 3), ("orl", 5, 10), ("vggface", 7, 2),
                ("paper_anchor", 9, 2)]


@pytest.mark.parametrize("name,n,K", EXPAND_CASES)
def test_expand_bit_exact(handle, name, n, K):
    w = _small(name, n, 40 if name == "orl" else 4, K)
    if name == "orl":
        w = dataclasses.replace(w, n_train=40)
    trx, _, _, _ = synth.make_dataset(w)
    trx = trx[:n]
    ker = synth.make_kernels(w, K)
    H = handle.expand(lb.arch_of(w, 1.0), _dev(trx), _dev(ker)).cpu().numpy()
    oa = _orc_arch(w)
    for k in range(K):
        u = orc.expand(oa, trx, ker[k])
        assert np.array_equal(H[k].astype(np.int64), u), (name, k)
        assert np.array_equal(H[k], u.astype(np.float32))


def _variant_arch_cases():
    F, D = lb.CONV_FULL, lb.CONV_DEPTHWISE
    return [
        # paper pool (4,2,1,cover_all) on the config-2/3 layer stacks: same F as the (2,2,0) reading
        ("mnist_paperpool", (28, 28, 1), [(F, 10, 3, 0, 4, 2, 1, 1), (F, 20, 3, 0, 4, 2, 1, 1)]),
        ("gtsrb_paperpool", (32, 32, 3), [(F, 16, 3, 0, 4, 2, 1, 1), (F, 32, 3, 0, 4, 2, 1, 1)]),
        # three layers, mixed types, relu, odd channel counts, 5x5 then 3x3, no pool in the middle
        ("three_layers", (19, 23, 2), [(F, 5, 5, 1, 2, 2, 0, 0), (D, 3, 3, 0, 1, 1, 0, 0), (F, 7, 3, 1, 3, 2, 1, 1)]),
        # Table II family (40,2,2) depthwise: F = 2560
        ("mnist_40_2_2", (28, 28, 1), [(D, 40, 3, 0, 4, 2, 1, 1), (D, 2, 3, 0, 4, 2, 1, 1), (D, 2, 3, 0, 4, 2, 1, 1)]),
        ("k7_single", (9, 8, 1), [(F, 2, 7, 0, 3, 3, 0, 1)]),
    ]


@pytest.mark.parametrize("name,shape,layers", _variant_arch_cases(), ids=[c[0] for c in _variant_arch_cases()])
def test_expand_variants_with_bias(handle, name, shape, layers):
    rng = np.random.default_rng(zlib.crc32(name.encode()))
    n, K = 6, 3
    x = rng.integers(0, 256, size=(n,) + shape, dtype=np.uint8)
    arch = lb.make_arch(*shape, layers, 1.0)
    nw, nb = lb.kernel_set_size(arch)
    ker = (rng.integers(0, 2, size=(K, nw)) * 2 - 1).astype(np.int8)
    bias = rng.integers(-300, 300, size=(K, nb)).astype(np.int32)
    oa = orc.make_arch(*shape, layers)
    F, _ = lb.feature_dim(arch)
    assert F == orc.feature_dim(oa)[0]
    for use_bias in (False, True):
        H = handle.expand(arch, _dev(x), _dev(ker), _dev(bias) if use_bias else None).cpu().numpy()
        for k in range(K):
            u = orc.expand(oa, x, ker[k], bias[k] if use_bias else None)
            assert np.array_equal(H[k].astype(np.int64), u), (name, use_bias, k)


def _tc_envelope_cases():
    F = lb.CONV_FULL
    return [
        # relu on both layers, odd channel counts, ragged image batch and candidate split
        ("relu2", (20, 24, 1), [(F, 6, 3, 1, 2, 2, 0, 0), (F, 9, 3, 1, 2, 2, 0, 0)], 23, 5),
        # single layer without pooling (one phase) and with 2x2 pooling
        ("one_layer_nopool", (16, 16, 3), [(F, 16, 3, 0, 1, 1, 0, 0)], 9, 4),
        ("one_layer_pool2", (18, 14, 2), [(F, 7, 3, 0, 2, 2, 0, 0)], 19, 3),
        # 5x5 kernels with 4x4 pooling (configs[3]'s family) on a non-square image
        ("k5_pool4", (24, 20, 2), [(F, 5, 5, 0, 4, 4, 0, 0)], 7, 6),
        # second layer without pooling and with more than 32 kernels
        ("l2_nopool_wide", (12, 12, 1), [(F, 3, 3, 0, 2, 2, 0, 0), (F, 40, 3, 0, 1, 1, 0, 0)], 11, 3),
        # 5x5 kernels in both layers (run-time tap loop of the layer-2 issuer)
        ("k5_k5", (16, 16, 1), [(F, 8, 5, 0, 2, 2, 0, 0), (F, 17, 5, 1, 2, 2, 0, 0)], 10, 3),
        # 4x4 pooling feeding a second layer
        ("pool4_then_pool2", (32, 32, 1), [(F, 4, 3, 0, 4, 4, 0, 0), (F, 12, 3, 0, 2, 2, 0, 0)], 13, 2),
        # many candidates over few images: candidate groups per CTA, last group ragged
        ("many_cands", (28, 28, 1), [(F, 10, 3, 0, 2, 2, 0, 0), (F, 20, 3, 0, 2, 2, 0, 0)], 50, 70),
    ]


@pytest.mark.parametrize("name,shape,layers,n,K", _tc_envelope_cases(), ids=[c[0] for c in _tc_envelope_cases()])
def test_expand_tensor_core_envelope(handle, name, shape, layers, n, K):
    """architectures inside the tcgen05 expander's envelope: the tensor-core kernel must be the one taken and its
    integers must equal the oracle's (and extreme pixels 0 / 255 must not overflow the int8 digits)."""
    rng = np.random.default_rng(zlib.crc32(name.encode()))
    x = rng.integers(0, 256, size=(n,) + shape, dtype=np.uint8)
    x[0] = 255
    x[-1] = 0
    arch = lb.make_arch(*shape, layers, 1.0)
    assert handle.expand_path(arch) == lb.EXPAND_TENSOR, name
    nw, _ = lb.kernel_set_size(arch)
    ker = (rng.integers(0, 2, size=(K, nw)) * 2 - 1).astype(np.int8)
    ker[0] = 1          # all +1: the largest layer-1 sums
    H = handle.expand(arch, _dev(x), _dev(ker)).cpu().numpy()
    oa = orc.make_arch(*shape, layers)
    for k in range(min(K, 6)):
        u = orc.expand(oa, x, ker[k])
        assert np.array_equal(H[k].astype(np.int64), u), (name, k)
    if K > 6:
        u = orc.expand(oa, x, ker[K - 1])
        assert np.array_equal(H[K - 1].astype(np.int64), u), (name, K - 1)


def test_expand_path_selection(handle):
    F, D = lb.CONV_FULL, lb.CONV_DEPTHWISE
    for name in ("tiny_mnist", "mnist", "gtsrb", "orl", "vggface"):
        assert handle.expand_path(lb.arch_of(synth.WORKLOADS[name], 1.0)) == lb.EXPAND_TENSOR, name
    assert handle.expand_path(lb.arch_of(synth.WORKLOADS["paper_anchor"], 1.0)) == lb.EXPAND_SIMT     # depthwise, cover_all
    assert handle.expand_path(lb.arch_of(synth.WORKLOADS["mnist"], 1.0), has_bias=True) == lb.EXPAND_SIMT
    assert handle.expand_path(lb.make_arch(28, 28, 1, [(F, 10, 3, 0, 4, 2, 1, 1)], 1.0)) == lb.EXPAND_SIMT  # overlapping pool
    assert handle.expand_path(lb.make_arch(28, 28, 1, [(F, 20, 3, 0, 2, 2, 0, 0), (F, 8, 3, 0, 2, 2, 0, 0)], 1.0)) == lb.EXPAND_SIMT


def test_expand_scaled_features(handle):
    w = _small("gtsrb", 17, 4, 2)
    trx, _, _, _ = synth.make_dataset(w)
    ker = synth.make_kernels(w, 2)
    s = np.float32(1.0 / 255.0)
    H = handle.expand(lb.arch_of(w, float(s)), _dev(trx), _dev(ker)).cpu().numpy().astype(np.float64)
    for k in range(2):
        ref = orc.expand(_orc_arch(w), trx, ker[k]).astype(np.float64) * float(s)
        z = ref == 0
        assert np.array_equal(H[k][z], ref[z])
        rel = np.abs(H[k][~z] - ref[~z]) / np.abs(ref[~z])
        assert rel.max() <= TOL_FEAT_REL


def _fro(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def _fit_case(handle, H, y, c, Creg, s, flags=0):
    K = H.shape[0]
    n, F = H.shape[1], H.shape[2]
    handle.ensure_workspace(lb.fit_workspace_bytes(n, F, c, K, flags))
    W, info = handle.elm_fit(_dev(H), _dev(y), c, Creg, h_scale=s, flags=flags)
    return W.cpu().numpy().astype(np.float64), info.cpu().numpy()


@pytest.mark.parametrize("n,F,c,flags", [(150, 70, 5, 0), (70, 150, 5, 0), (130, 130, 3, 0), (257, 129, 11, lb.FORCE_DUAL),
                                         (90, 200, 7, lb.FORCE_PRIMAL), (64, 64, 2, 0), (3, 2, 2, 0)])
def test_fit_matches_oracle_general_fp32(handle, n, F, c, flags):
    rng = np.random.default_rng(n * 1000 + F)
    K = 3
    H = rng.standard_normal((K, n, F)).astype(np.float32)
    y = rng.integers(0, c, size=n).astype(np.int32)
    y[:c] = np.arange(c) if n >= c else y[:c]
    W, info = _fit_case(handle, H, y, c, 10.0, 1.0, flags)
    assert (info == 0).all()
    for k in range(K):
        Wo, inf, br = orc.elm_fit(H[k].astype(np.float64), y, c, 10.0)
        assert inf == 0
        assert _fro(W[k], Wo) <= TOL_W_FRO
        assert _fro(W[k], Wo) <= 1e-5     # what the fp64 path actually delivers (fp32 rounding of W)


@pytest.mark.parametrize("n,F,c,panel,integer", [(1500, 700, 5, 128, False), (2100, 1100, 12, 256, True),
                                                  (900, 2000, 7, 192, False), (1300, 577, 3, 64, True)])
def test_fit_tensor_core_solver(handle, n, F, c, panel, integer):
    """LBCNN_SOLVER_MIXED: the trailing updates of the blocked Cholesky as int8 digit products on tcgen05 (chol_tc.cu).
    Ragged dimensions (not multiples of 64 / 128 / the panel), primal and dual, well- and ill-conditioned (integer
    features with a common mode, cond ~ 1e6 like the expander's output): W against the oracle within north_star's
    1e-3 and against the all-fp64 solver within 1e-4."""
    rng = np.random.default_rng(n + F)
    K = 2
    if integer:
        base = rng.integers(0, 4000, size=(K, 1, F))
        H = (base + rng.integers(-300, 300, size=(K, n, F))).astype(np.float32)
        s, Creg, flags = 1.0 / 255.0, 1e4, lb.H_INTEGER
    else:
        H = rng.standard_normal((K, n, F)).astype(np.float32)
        s, Creg, flags = 1.0, 10.0, 0
    y = rng.integers(0, c, size=n).astype(np.int32)
    Hd, yd = _dev(H), _dev(y)
    handle.set_workspace(None)
    handle.ensure_workspace(lb.fit_workspace_bytes(n, F, c, K, flags))
    try:
        handle.set_option(lb.OPT_SOLVER, lb.SOLVER_MIXED)
        handle.set_option(lb.OPT_PANEL, panel)
        handle.set_option(lb.OPT_MID_PANEL, {256: 128, 192: 64}.get(panel, 0))     # three levels on two of the cases
        W_tc, info_tc = handle.elm_fit(Hd, yd, c, Creg, h_scale=s, flags=flags)
        handle.set_option(lb.OPT_SOLVER, lb.SOLVER_FP64)
        W_64, info_64 = handle.elm_fit(Hd, yd, c, Creg, h_scale=s, flags=flags)
        torch.cuda.synchronize()
    finally:
        handle.set_option(lb.OPT_SOLVER, lb.SOLVER_AUTO)
        handle.set_option(lb.OPT_PANEL, 1024)
        handle.set_option(lb.OPT_MID_PANEL, 256)
    assert (info_tc.cpu().numpy() == 0).all() and (info_64.cpu().numpy() == 0).all()
    sc = float(np.float32(s))
    for k in range(K):
        a, b = W_tc[k].cpu().numpy().astype(np.float64), W_64[k].cpu().numpy().astype(np.float64)
        assert _fro(a, b) <= 1e-4, _fro(a, b)
        Wo, inf, _ = orc.elm_fit(H[k].astype(np.float64) * sc, y, c, Creg)
        assert inf == 0 and _fro(a, Wo) <= TOL_W_FRO, _fro(a, Wo)


def test_fit_worked_example(handle):
    # tests/golden/worked_examples.txt [elm_small]: H=[[1,0],[0,1],[1,1]], labels [0,1,0], C=1 -> W=[[.625,-.125],[.125,.375]]
    H = np.array([[[1, 0], [0, 1], [1, 1]]], dtype=np.float32)
    y = np.array([0, 1, 0], dtype=np.int32)
    for flags in (lb.FORCE_PRIMAL, lb.FORCE_DUAL, 0):
        W, info = _fit_case(handle, H, y, 2, 1.0, 1.0, flags)
        assert info[0] == 0
        assert np.allclose(W[0], [[0.625, -0.125], [0.125, 0.375]], atol=1e-7)
    # scale identity W(sH, C) = W(H, C s^2)/s, here through h_scale
    W2, _ = _fit_case(handle, H, y, 2, 4.0, 0.5)
    assert np.allclose(W2[0], 2.0 * np.array([[0.625, -0.125], [0.125, 0.375]]), atol=1e-6)


def test_fit_failure_is_reported_per_candidate(handle):
    rng = np.random.default_rng(5)
    H = rng.standard_normal((3, 40, 8)).astype(np.float32)
    H[1, 3, 2] = np.nan
    y = rng.integers(0, 3, size=40).astype(np.int32)
    W, info = _fit_case(handle, H, y, 3, 1.0, 1.0)
    assert info[0] == 0 and info[2] == 0 and info[1] > 0
    # the oracle stops at the same pivot: the NaN sits in feature 2, so pivot 2 is the first that is not > 0
    _, inf_o, br = orc.elm_fit(H[1].astype(np.float64), y, 3, 1.0)
    assert br == 1 and inf_o == 3 and info[1] == inf_o
    Wd, infod = _fit_case(handle, H, y, 3, 1.0, 1.0, lb.FORCE_DUAL)          # dual: the NaN sits in sample 3
    _, inf_od, brd = orc.elm_fit(H[1].astype(np.float64), y, 3, 1.0, force_branch=2)
    assert brd == 2 and inf_od == 4 and infod[1] == inf_od and infod[0] == 0 and infod[2] == 0
    Wo, _, _ = orc.elm_fit(H[2].astype(np.float64), y, 3, 1.0)
    assert _fro(W[2], Wo) <= 1e-5


def test_score_matches_oracle_and_ties(handle):
    rng = np.random.default_rng(11)
    K, n, F, c = 2, 203, 97, 70
    H = rng.integers(-50, 50, size=(K, n, F)).astype(np.float32)
    W = rng.standard_normal((K, F, c)).astype(np.float32)
    y = rng.integers(0, c, size=n).astype(np.int32)
    pred, corr = handle.elm_score(_dev(H), _dev(W), _dev(y), h_scale=0.25)
    pred, corr = pred.cpu().numpy(), corr.cpu().numpy()
    for k in range(K):
        po, co, _ = orc.elm_score(H[k].astype(np.float64) * 0.25, W[k].astype(np.float64), y)
        assert np.array_equal(pred[k], po)
        assert corr[k] == co
    # exact ties -> lowest class index; all-zero W -> class 0
    Wz = np.zeros((1, F, c), dtype=np.float32)
    pz, _ = handle.elm_score(_dev(H[:1]), _dev(Wz))
    assert (pz.cpu().numpy() == 0).all()
    Wt = np.zeros((1, F, c), dtype=np.float32)
    Wt[0, :, 65] = 1.0
    Wt[0, :, 3] = 1.0
    Hp = np.abs(H[:1]) + 1
    pt, _ = handle.elm_score(_dev(Hp), _dev(Wt))
    assert (pt.cpu().numpy() == 3).all()


@pytest.mark.parametrize("K,n,F,c,amax", [(2, 203, 96, 70, 50), (3, 1000, 980, 10, 200000), (1, 300, 2048, 43, 900000),
                                          (2, 517, 260, 128, 6000), (1, 129, 8, 2, 3)])
def test_score_tensor_core_equals_fp64_argmax(handle, K, n, F, c, amax):
    """LBCNN_SCORER_TENSOR (score_tc.cu): int8 digit products on tcgen05 + exact fp64 re-evaluation of the rows inside
    the error bound.  Labels must equal the oracle's fp64 argmax ONE BY ONE -- including exact ties (lowest index), rows
    that hold a non-integer or an out-of-range feature, an all-zero W, ragged n and F not a multiple of 64."""
    rng = np.random.default_rng(K * 1000 + F)
    base = rng.integers(0, amax // 2 + 1, size=(K, 1, F))
    H = (base + rng.integers(-(amax // 2), amax // 2 + 1, size=(K, n, F))).astype(np.float32)
    H[0, 3, 1] = 0.5                     # not an integer
    H[0, 5, 2] = 9.0e6                   # outside three balanced radix-256 digits
    H[0, 7, :] = 0.0
    W = (rng.standard_normal((K, F, c)) * rng.uniform(1e-4, 1.0, size=(K, 1, c))).astype(np.float32)
    W[0, :, c - 1] = W[0, :, 0]          # exact ties between class 0 and the last class: class 0 must win
    y = rng.integers(0, c, size=n).astype(np.int32)
    hs = 1.0 / 255.0
    handle.set_workspace(None)
    handle.ensure_workspace(lb.score_workspace_bytes(n, F, c, K))
    try:
        handle.set_option(lb.OPT_SCORER, lb.SCORER_TENSOR)
        pred, corr = handle.elm_score(_dev(H), _dev(W), _dev(y), h_scale=hs)
        Wz = np.zeros((1, F, c), dtype=np.float32)
        pz, _ = handle.elm_score(_dev(H[:1]), _dev(Wz))
        handle.set_option(lb.OPT_SCORER, lb.SCORER_FP64)
        pred64, corr64 = handle.elm_score(_dev(H), _dev(W), _dev(y), h_scale=hs)
        torch.cuda.synchronize()
    finally:
        handle.set_option(lb.OPT_SCORER, lb.SCORER_AUTO)
    pred, corr = pred.cpu().numpy(), corr.cpu().numpy()
    assert (pz.cpu().numpy() == 0).all()
    sc = float(np.float32(hs))
    for k in range(K):
        po, co, margin = orc.elm_score(H[k].astype(np.float64) * sc, W[k].astype(np.float64), y, want_margin=True)
        differ = np.nonzero(pred[k] != po)[0]
        # the only admissible differences are fp64 rounding-order effects at margins ~1e-16 of the logits
        assert len(differ) == 0 or np.all(margin[differ] <= 1e-12 * np.abs(H[k].astype(np.float64) * sc).sum(1)[differ].max()), (k, differ[:10], margin[differ][:10])
        assert corr[k] == int((pred[k] == y).sum())
    assert torch.equal(torch.from_numpy(pred), pred64.cpu()) or (pred != pred64.cpu().numpy()).mean() < 1e-3
    assert (pred[0] != c - 1).all() or c == 2          # ties resolved to the lower index


@pytest.mark.parametrize("name,ntr,nte,K,bits", [("mnist", 1500, 700, 3, 8), ("gtsrb", 2600, 900, 2, 8), ("orl", 280, 120, 4, 6),
                                                  ("tiny_mnist", 2000, 500, 3, 4)])
def test_quantised_output_layer_matches_oracle(handle, name, ntr, nte, K, bits):
    """SURVEY.md 8(f)-2 ("weights represented as 8 bits integers"; R16): lbcnn_quantize_output_layer
    must reproduce the oracle's integers and scale BIT-EXACTLY, and lbcnn_elm_score_q (exact integer logits on the tensor
    pipe) the oracle's labels ONE BY ONE with identical counts -- integer work, so no tolerance."""
    w = _small(name, ntr, nte, K)
    trx, try_, tex, tey = synth.make_dataset(w)
    ker = synth.make_kernels(w)
    W, _, _, info = _staged(handle, w, trx, try_, tex, tey, ker)
    assert (info == 0).all()
    W32 = W.astype(np.float32)
    Hte = handle.expand(lb.arch_of(w, 1.0), _dev(tex), _dev(ker))
    Wq, scale = handle.quantize_output_layer(_dev(W32), bits)
    pred, corr = handle.elm_score_q(Hte, Wq, _dev(tey))
    torch.cuda.synchronize()
    Wq, scale, pred, corr = Wq.cpu().numpy(), scale.cpu().numpy(), pred.cpu().numpy(), corr.cpu().numpy()
    oa = _orc_arch(w)
    for k in range(K):
        qo, so = orc.quantize_output_layer(W32[k], bits)
        assert np.array_equal(Wq[k], qo), k
        assert scale[k] == so
        po, co, logits = orc.elm_score_q(orc.expand(oa, tex, ker[k]), qo, tey)
        assert np.array_equal(pred[k], po), (k, np.nonzero(pred[k] != po)[0][:10])
        assert corr[k] == co
    # constructed ties and a row with a non-integer feature (evaluated in fp64 by the second kernel)
    H2 = Hte[:1].clone()
    H2[0, 1, 0] += 0.5
    q2 = Wq[:1].copy()
    q2[0, :, w.n_classes - 1] = q2[0, :, 0]
    p2, _ = handle.elm_score_q(H2, _dev(q2))
    p2 = p2.cpu().numpy()[0]
    ref = (H2[0].cpu().numpy().astype(np.float64) @ q2[0].astype(np.float64))
    assert (p2 != w.n_classes - 1).all()
    rows = np.arange(len(p2)) != 1
    assert np.array_equal(p2[rows], np.argmax(ref, axis=1)[rows])
    assert p2[1] == int(np.argmax(ref[1]))


def test_genetic_generator_bit_exact_and_improves(handle):
    """lbcnn_evolve_candidates must reproduce the oracle's next
    generation byte for byte (ties in the ranking, a failed candidate, elites, several mutation rates), and a search driven
    by it keeps its best accuracy from generation to generation (elitism) on the tiny config."""
    rng = np.random.default_rng(33)
    for K, nw, elite, ppm, seed, gen in [(24, 300, 4, 20000, 7, 2), (7, 1890, 1, 0, 123456789012345, 0), (64, 37, 0, 1000000, 1, 9),
                                         (130, 513, 130, 5000, 2, 1)]:
        ker = (rng.integers(0, 2, size=(K, nw)) * 2 - 1).astype(np.int8)
        acc = rng.integers(50, 60, size=K).astype(np.float32) / 100.0          # many exact ties
        acc[K // 2] = -1.0
        nxt = handle.evolve_candidates(_dev(ker), _dev(acc), elite, ppm, seed, gen).cpu().numpy()
        ref, _, _ = orc.evolve_candidates(ker, acc, elite, ppm, seed, gen)
        assert np.array_equal(nxt, ref), (K, nw)
    # a three-generation search on configs[0]: elitism keeps the running best, children are evaluated by the same driver
    w = synth.WORKLOADS["tiny_mnist"]
    trx, try_, tex, tey = synth.make_dataset(w)
    ker = _dev(synth.make_kernels(w))
    arch = lb.arch_of(w)
    data = (_dev(trx), _dev(try_), _dev(tex), _dev(tey))
    best = []
    for g in range(3):
        handle.set_workspace(None)
        handle.ensure_workspace(lb.workspace_bytes(arch, w.n_train, w.n_test, w.n_classes, w.n_cand)[0])
        out = handle.search_candidates(arch, *data, w.n_classes, w.C, ker)
        acc = out["acc"].clone()
        best.append(float(acc.max()))
        ker = handle.evolve_candidates(ker, acc, 2, 30000, 99, g)
    assert best[1] >= best[0] and best[2] >= best[1]


@pytest.mark.parametrize("name,ntr,nte,epochs,batch", [("mnist", 1500, 700, 3, 128), ("gtsrb", 900, 300, 2, 100), ("tiny_mnist", 333, 100, 4, 64)])
def test_refine_output_layer_matches_oracle(handle, name, ntr, nte, epochs, batch):
    """SURVEY.md 8(f)-4 (PAPER.md:98 Cell 10; R18 = SPEC.md:324, 355): softmax cross-entropy + Adam on the output
    layer, starting from the ELM fit, features from the frozen binary kernels.  fp64 on both sides: the refined W must
    match the oracle's within north_star's 1e-3 (it does to ~1e-9), the per-epoch losses to 1e-6, labels one by one;
    epochs = 0 is the identity; a ragged last batch on purpose."""
    w = _small(name, ntr, nte, 1)
    trx, try_, tex, tey = synth.make_dataset(w)
    ker = synth.make_kernels(w)
    W0, _, _, info = _staged(handle, w, trx, try_, tex, tey, ker)
    assert info[0] == 0
    a1 = lb.arch_of(w, 1.0)
    s = float(np.float32(w.feature_scale))
    Htr = handle.expand(a1, _dev(trx), _dev(ker))[0].contiguous()
    Hte = handle.expand(a1, _dev(tex), _dev(ker))
    W0f = _dev(W0[0].astype(np.float32))
    Wn, loss = handle.refine_output_layer(Htr, _dev(try_), W0f, epochs=epochs, batch=batch, lr=1e-3, seed=5, h_scale=s)
    Wsame, _ = handle.refine_output_layer(Htr, _dev(try_), W0f, epochs=0, batch=batch, h_scale=s)
    torch.cuda.synchronize()
    assert torch.equal(Wsame, W0f)
    oa = _orc_arch(w)
    Uo = orc.expand(oa, trx, ker[0]).astype(np.float64)
    Wo, lo = orc.refine_output_layer(Uo, try_, W0[0].astype(np.float32).astype(np.float64), epochs, batch, 1e-3, seed=5, h_scale=s)
    err = _fro(Wn.cpu().numpy().astype(np.float64), Wo)
    assert err <= TOL_W_FRO and err <= 1e-5, err
    assert np.allclose(loss.cpu().numpy(), lo, rtol=1e-5, atol=1e-7)      # (whether the loss falls at this lr is the recipe's business)
    pred, _ = handle.elm_score(Hte, Wn[None].contiguous(), _dev(tey), h_scale=s)
    po, _, _ = orc.elm_score(orc.expand(oa, tex, ker[0]).astype(np.float64) * s, Wo, tey)
    assert (pred.cpu().numpy()[0] == po).mean() >= TOL_LABEL_AGREE


def test_genetic_generator_nan_accuracy(handle):
    """A NaN accuracy (0 / 0 from an empty test set upstream, or garbage passed in) ranks as minus infinity (R17): the
    ranks stay a permutation, the elites are real candidates and the result equals the oracle's byte for byte."""
    rng = np.random.default_rng(77)
    K, nw = 40, 129
    ker = (rng.integers(0, 2, size=(K, nw)) * 2 - 1).astype(np.int8)
    acc = rng.integers(50, 60, size=K).astype(np.float32) / 100.0
    acc[[3, 17, 18, 39]] = np.nan
    acc[5] = -1.0
    for elite in (K, 6):
        ref, _, order = orc.evolve_candidates(ker, acc, elite, 10000, 4, 3)
        assert order.tolist()[-5:] == [5, 3, 17, 18, 39]
        nxt = handle.evolve_candidates(_dev(ker), _dev(acc), elite, 10000, 4, 3).cpu().numpy()
        assert np.array_equal(nxt, ref)
        nxt = handle.evolve_candidates_static(_dev(ker), _dev(acc), elite, 10000, 4, 3).cpu().numpy()
        assert np.array_equal(nxt, ref)


def test_refine_adam_worked_example_and_many_epochs(handle):
    """(1) The hand-worked two Adam steps of tests/golden/worked_examples.txt [adam_two_steps] (R18) on the GPU: W after
    step 2 = 0.19958968129158736 on the diagonal, reached across epochs and inside one epoch.  W comes back as fp32.
    (2) More epochs than F * n_classes rounded up to a block (the loss accumulators beyond the weight count must start at
    zero): 300 epochs on a 2 x 2 layer against the oracle, twice in the same workspace."""
    w2 = 0.19958968129158736
    want = np.array([[w2, -w2], [-w2, w2]])
    H = torch.eye(2, device="cuda"); y = torch.tensor([0, 1], dtype=torch.int32, device="cuda"); W0 = torch.zeros((2, 2), device="cuda")
    W, loss = handle.refine_output_layer(H, y, W0, epochs=2, batch=2, lr=0.1, seed=3)
    assert np.allclose(W.cpu().numpy(), want, rtol=0, atol=2e-8)
    assert np.allclose(loss.cpu().numpy(), [0.6931471805599453, 0.5981388729829197], rtol=0, atol=1e-7)
    H4 = torch.cat([H, H]).contiguous(); y4 = torch.cat([y, y]).contiguous()
    W, _ = handle.refine_output_layer(H4, y4, W0, epochs=1, batch=2, lr=0.1, seed=3)
    assert np.allclose(W.cpu().numpy(), want, rtol=0, atol=2e-8)
    rng = np.random.default_rng(9)
    Hn = rng.normal(size=(33, 2)).astype(np.float32); yn = rng.integers(0, 2, size=33).astype(np.int32)
    for rep in range(2):
        Wg, lg = handle.refine_output_layer(_dev(Hn), _dev(yn), W0, epochs=300, batch=16, lr=1e-2, seed=rep)
        Wo, lo = orc.refine_output_layer(Hn.astype(np.float64), yn, np.zeros((2, 2)), 300, 16, 1e-2, seed=rep)
        assert np.allclose(lg.cpu().numpy(), lo, rtol=1e-5, atol=1e-7)
        assert _fro(Wg.cpu().numpy().astype(np.float64), Wo) <= 1e-5


def _search_both(handle, w, budget=None):
    trx, try_, tex, tey = synth.make_dataset(w)
    ker = synth.make_kernels(w)
    arch = lb.arch_of(w)
    full, mn = lb.workspace_bytes(arch, w.n_train, w.n_test, w.n_classes, w.n_cand, budget or 0)
    handle.set_workspace(None)
    handle.ensure_workspace(full)
    out = handle.search_candidates(arch, _dev(trx), _dev(try_), _dev(tex), _dev(tey), w.n_classes, w.C, _dev(ker))
    torch.cuda.synchronize()
    ref = orc.search(_orc_arch(w), trx, try_, tex, tey, w.n_classes, w.C, ker, feature_scale=w.feature_scale, keep=True)
    return {k: (v.cpu().numpy() if v is not None else None) for k, v in out.items()}, ref


def _staged(handle, w, trx, try_, tex, tey, ker_sel):
    """the three stand-alone entry points on the selected candidates, exactly as the driver chains them (integer
    features, h_scale, LBCNN_H_INTEGER): returns (W [k][F][c] float64, pred [k][n_test], correct [k], info [k])."""
    a1 = lb.arch_of(w, 1.0)
    s = float(np.float32(w.feature_scale))
    kd = _dev(ker_sel)
    Htr = handle.expand(a1, _dev(trx), kd)
    Hte = handle.expand(a1, _dev(tex), kd)
    F = Htr.shape[2]
    handle.ensure_workspace(lb.fit_workspace_bytes(w.n_train, F, w.n_classes, len(ker_sel), lb.H_INTEGER))
    W, info = handle.elm_fit(Htr, _dev(try_), w.n_classes, w.C, h_scale=s, flags=lb.H_INTEGER)
    pred, corr = handle.elm_score(Hte, W, _dev(tey), h_scale=s)
    torch.cuda.synchronize()
    return W.cpu().numpy().astype(np.float64), pred.cpu().numpy(), corr.cpu().numpy(), info.cpu().numpy()


def _check_labels_and_W(handle, w, got_correct, ref_W, ref_pred, cands, data=None):
    """predicted labels ONE BY ONE and W of every candidate in `cands` against the oracle's; the staged calls are tied
    to the driver's result through the per-candidate correct counts, which must be identical."""
    trx, try_, tex, tey = data if data is not None else synth.make_dataset(w)
    ker = synth.make_kernels(w)
    cands = sorted(set(int(k) for k in cands))
    W, pred, corr, info = _staged(handle, w, trx, try_, tex, tey, ker[cands])
    assert (info == 0).all()
    for j, k in enumerate(cands):
        assert int(corr[j]) == int(got_correct[k]), ("driver and staged calls disagree", k)
        agree = float((pred[j] == ref_pred[k]).mean())
        assert agree >= TOL_LABEL_AGREE, (k, agree)
        assert _fro(W[j], ref_W[k]) <= TOL_W_FRO, (k, _fro(W[j], ref_W[k]))
        co = int((ref_pred[k] == tey).sum())
        assert abs(int(corr[j]) - co) / float(w.n_test) * 100.0 <= TOL_ACC_PP


def _check_search(handle, w, got, ref):
    K = w.n_cand
    assert (got["info"] == 0).all() and (ref["info"] == 0).all()
    assert (np.abs(got["acc"].astype(np.float64) - ref["acc"]) * 100.0 <= TOL_ACC_PP).all()
    assert np.array_equal(got["acc"], (got["correct"].astype(np.float64) / w.n_test).astype(np.float32))
    b, wst = int(got["best"][0]), int(got["best"][1])
    assert b == int(np.argmax(got["correct"])) and wst == int(np.argmin(got["correct"]))     # first max / first min
    if b != ref["best"]:
        assert abs(ref["acc"][b] - ref["acc"][ref["best"]]) * 100.0 <= TOL_ACC_PP      # near-tie only
    if wst != ref["worst"]:
        assert abs(ref["acc"][wst] - ref["acc"][ref["worst"]]) * 100.0 <= TOL_ACC_PP
    assert _fro(got["W_best"].astype(np.float64), ref["W"][b]) <= TOL_W_FRO
    assert K == len(ref["acc"])
    # labels one by one and W for the best, the worst, the first and the last candidate (at least two per config)
    _check_labels_and_W(handle, w, got["correct"], ref["W"], ref["pred"], {b, wst, 0, K - 1})


SEARCH_CASES = [("tiny_mnist", None, None, None), ("mnist", 1500, 700, 5), ("gtsrb", 2600, 500, 3),
                ("orl", 280, 120, 12), ("vggface", 900, 300, 2), ("paper_anchor", 300, 200, 2)]


@pytest.mark.parametrize("name,ntr,nte,K", SEARCH_CASES, ids=[c[0] for c in SEARCH_CASES])
def test_search_matches_oracle(handle, name, ntr, nte, K):
    w = synth.WORKLOADS[name] if ntr is None else _small(name, ntr, nte, K)
    got, ref = _search_both(handle, w)
    _check_search(handle, w, got, ref)


def test_search_with_bias_matches_oracle(handle):
    """a bias is an arbitrary int32 added before the pooling (PAPER.md:51, 53 `b=bias`; R14): the driver must
    leave the digit envelope of the exact tensor-core Gram aside (bias is not part of the feature bound) and still
    match the oracle -- accuracies, labels through the counts, W of the best candidate."""
    w = _small("mnist", 700, 300, 4)
    trx, try_, tex, tey = synth.make_dataset(w)
    ker = synth.make_kernels(w)
    arch = lb.arch_of(w)
    _, nb = lb.kernel_set_size(arch)
    rng = np.random.default_rng(77)
    bias = rng.integers(-3000, 3000, size=(w.n_cand, nb)).astype(np.int32)
    handle.set_workspace(None)
    handle.ensure_workspace(lb.workspace_bytes(arch, w.n_train, w.n_test, w.n_classes, w.n_cand)[0])
    out = handle.search_candidates(arch, _dev(trx), _dev(try_), _dev(tex), _dev(tey), w.n_classes, w.C, _dev(ker), _dev(bias))
    got = {k: v.cpu().numpy() for k, v in out.items()}
    ref = orc.search(_orc_arch(w), trx, try_, tex, tey, w.n_classes, w.C, ker, feature_scale=w.feature_scale, bias=bias, keep=True)
    assert (got["info"] == 0).all() and (ref["info"] == 0).all()
    assert (np.abs(got["acc"].astype(np.float64) - ref["acc"]) * 100.0 <= TOL_ACC_PP).all()
    b = int(got["best"][0])
    assert _fro(got["W_best"].astype(np.float64), ref["W"][b]) <= TOL_W_FRO
    # labels one by one through the staged entry points with the same bias (general fp32 H: flags = 0)
    a1 = lb.arch_of(w, 1.0)
    s = float(np.float32(w.feature_scale))
    Htr = handle.expand(a1, _dev(trx), _dev(ker), _dev(bias))
    Hte = handle.expand(a1, _dev(tex), _dev(ker), _dev(bias))
    handle.ensure_workspace(lb.fit_workspace_bytes(w.n_train, Htr.shape[2], w.n_classes, w.n_cand, 0))
    W, info = handle.elm_fit(Htr, _dev(try_), w.n_classes, w.C, h_scale=s, flags=0)
    pred, corr = handle.elm_score(Hte, W, _dev(tey), h_scale=s)
    assert np.array_equal(corr.cpu().numpy(), got["correct"])
    for k in range(w.n_cand):
        assert (pred[k].cpu().numpy() == ref["pred"][k]).mean() >= TOL_LABEL_AGREE
        assert _fro(W[k].cpu().numpy().astype(np.float64), ref["W"][k]) <= TOL_W_FRO
    # features handed to the fit with the LBCNN_H_INTEGER promise broken (candidate 1: one value outside three balanced
    # radix-256 digits, |u| <= 8355711) are reported, not silently wrapped
    Htr[1, 5, 7] = 8355712.0
    handle.ensure_workspace(lb.fit_workspace_bytes(w.n_train, Htr.shape[2], w.n_classes, w.n_cand, lb.H_INTEGER))
    _, info_i = handle.elm_fit(Htr, _dev(try_), w.n_classes, w.C, h_scale=s, flags=lb.H_INTEGER)
    info_i = info_i.cpu().numpy()
    assert info_i[1] == -1 and info_i[0] == 0 and info_i[2] == 0 and info_i[3] == 0


def test_search_is_deterministic_run_to_run(handle):
    """the tensor-core kernels carry hand-rolled mbarrier pipelines and generic -> async proxy hand-offs; a race would
    show as run-to-run differences.  Five runs of configs[0] and of a reduced configs[1] must be bit-identical."""
    for w in (synth.WORKLOADS["tiny_mnist"], _small("mnist", 900, 333, 9)):
        trx, try_, tex, tey = synth.make_dataset(w)
        ker = synth.make_kernels(w)
        arch = lb.arch_of(w)
        handle.set_workspace(None)
        handle.ensure_workspace(lb.workspace_bytes(arch, w.n_train, w.n_test, w.n_classes, w.n_cand)[0])
        args = (arch, _dev(trx), _dev(try_), _dev(tex), _dev(tey), w.n_classes, w.C, _dev(ker))
        first = {k: v.clone() for k, v in handle.search_candidates(*args).items()}
        for _ in range(4):
            again = handle.search_candidates(*args)
            for k in first:
                assert torch.equal(first[k], again[k]), k


@pytest.mark.parametrize("name,ntr,nte,K,rows", [("mnist", 1500, 700, 5, 400), ("gtsrb", 2600, 500, 3, 1000),
                                                  ("tiny_mnist", 2000, 500, 8, 300), ("vggface", 8300, 300, 2, 4096)])
def test_streamed_search_equals_resident(handle, name, ntr, nte, K, rows):
    """LBCNN_OPT_STREAM_ROWS ("limited GPU-RAM"): the train set passes through
    the expander in chunks whose exact integer Grams and right-hand sides add up, the test set is scored chunk by chunk;
    H of the whole set never exists.  Everything is exact integer arithmetic below 2^53, so the result must be
    BIT-IDENTICAL to the resident search -- and the workspace must be smaller (ragged last chunks on purpose)."""
    w = _small(name, ntr, nte, K)
    trx, try_, tex, tey = synth.make_dataset(w)
    ker = synth.make_kernels(w)
    arch = lb.arch_of(w)
    args = (arch, _dev(trx), _dev(try_), _dev(tex), _dev(tey), w.n_classes, w.C, _dev(ker))
    full = lb.workspace_bytes(arch, w.n_train, w.n_test, w.n_classes, w.n_cand, handle=handle)[0]
    handle.set_workspace(None)
    handle.ensure_workspace(full)
    a = {k: v.clone() for k, v in handle.search_candidates(*args).items()}
    try:
        handle.set_option(lb.OPT_STREAM_ROWS, rows)
        small = lb.workspace_bytes(arch, w.n_train, w.n_test, w.n_classes, w.n_cand, handle=handle)[0]
        assert small < full
        handle.set_workspace(None)
        handle.ensure_workspace(small)
        b = handle.search_candidates(*args)
        torch.cuda.synchronize()
    finally:
        handle.set_option(lb.OPT_STREAM_ROWS, 0)
    for k in a:
        assert torch.equal(a[k], b[k]), k
    assert (b["info"].cpu().numpy() == 0).all()
    handle.set_workspace(None)
    if name != "vggface":      # the streamed result against the ORACLE, not only against the resident CUDA search
        ref = orc.search(_orc_arch(w), trx, try_, tex, tey, w.n_classes, w.C, ker, feature_scale=w.feature_scale, keep=True)
        _check_search(handle, w, {k: v.cpu().numpy() for k, v in b.items()}, ref)


def test_streamed_search_beyond_the_int32_chunk_bound(handle):
    """N_train above 43690 (the exact Gram's int32 bound per launch; the paper's own case is the full 60000 of MNIST,
    PAPER.md:29, 104): LBCNN_OPT_STREAM_ROWS must still stream -- the bound is on the chunk, not on N -- and a request for
    chunks longer than the bound is served with chunks of the bound.  Checked against the oracle; that it really streamed is
    shown by the phase record (one Gram bracket per chunk, no separate right-hand side) and the int8 operation counter."""
    w = _small("tiny_mnist", 45000, 700, 3)
    trx, try_, tex, tey = synth.make_dataset(w)
    ker = synth.make_kernels(w)
    arch = lb.arch_of(w)
    F = lb.feature_dim(arch)[0]
    args = (arch, _dev(trx), _dev(try_), _dev(tex), _dev(tey), w.n_classes, w.C, _dev(ker))
    ref = orc.search(_orc_arch(w), trx, try_, tex, tey, w.n_classes, w.C, ker, feature_scale=w.feature_scale, keep=True)
    resident_H = w.n_cand * w.n_train * F * 4
    try:
        for rows, chunks in ((20000, 3), (44000, 2)):       # 44000 > 43690: served as 43690 + 1310
            handle.set_option(lb.OPT_STREAM_ROWS, rows)
            small = lb.workspace_bytes(arch, w.n_train, w.n_test, w.n_classes, w.n_cand, handle=handle)[0]
            if rows == 20000:
                assert small < resident_H, (rows, small, resident_H)
            handle.set_workspace(None)
            handle.ensure_workspace(small)
            handle.op_stats()
            handle.set_profiling(True)
            got = handle.search_candidates(*args)
            ph = handle.phase_times()
            handle.set_profiling(False)
            # one Gram bracket per chunk of samples, no separate right-hand-side phase, and the int8 Gram counter moved:
            # the streamed tensor-core plan ran, not the resident fp64 one
            assert ph["gram"][1] == chunks and ph["rhs"][1] == 0, ph
            assert handle.op_stats()["gram_int8_tmac"] > 0
            _check_search(handle, w, {k: v.cpu().numpy() for k, v in got.items()}, ref)
    finally:
        handle.set_option(lb.OPT_STREAM_ROWS, 0)
        handle.set_workspace(None)


@pytest.mark.parametrize("name,ntr,nte,K", [("orl", 280, 120, 16), ("vggface", 700, 300, 3), ("paper_anchor", 300, 200, 2)])
def test_dual_branch_kernel_trick_equals_explicit_w(handle, name, ntr, nte, K):
    """dual branch (F >= N): by default the driver scores through the cross-Gram -- logits =
    (H_te H^T)(H H^T + I/C)^-1 T out of the factorisation's appended rows, W only for the best candidate; with
    LBCNN_OPT_DUAL_TRICK = 0 it forms W = H^T Z for every candidate and scores H_te W.  Same mathematics: identical
    counts, best / worst, and W_best equal up to the rounding order of its fp64 sums."""
    w = _small(name, ntr, nte, K)
    trx, try_, tex, tey = synth.make_dataset(w)
    ker = synth.make_kernels(w)
    arch = lb.arch_of(w)
    handle.set_workspace(None)
    handle.ensure_workspace(lb.workspace_bytes(arch, w.n_train, w.n_test, w.n_classes, w.n_cand)[0])
    args = (arch, _dev(trx), _dev(try_), _dev(tex), _dev(tey), w.n_classes, w.C, _dev(ker))
    a = {k: v.clone() for k, v in handle.search_candidates(*args).items()}
    try:
        handle.set_option(lb.OPT_DUAL_TRICK, 0)
        b = handle.search_candidates(*args)
        torch.cuda.synchronize()
    finally:
        handle.set_option(lb.OPT_DUAL_TRICK, 1)
    for k in ("acc", "correct", "info", "best"):
        assert torch.equal(a[k], b[k]), k
    assert _fro(a["W_best"].cpu().numpy().astype(np.float64), b["W_best"].cpu().numpy().astype(np.float64)) <= 1e-6


@pytest.mark.parametrize("name,ntr,nte,K", [("orl", 280, 120, 16), ("vggface", 700, 300, 5)])
def test_dual_branch_chunked_equals_unchunked(handle, name, ntr, nte, K):
    """The decisions of a dual-branch search (correct[], acc, info, best / worst) must not depend on how much workspace the
    caller gave: the kernel-trick scoring is taken chunk by chunk as well, and the best candidate -- whose chunk may be gone by
    then -- is fitted once more on its own for W_best.  W_best then comes from the explicit W = H^T Z instead of the
    factorisation's rows: equal up to the rounding order of fp64 sums.  Both runs against the oracle too."""
    w = _small(name, ntr, nte, K)
    arch = lb.arch_of(w)
    full, mn = lb.workspace_bytes(arch, w.n_train, w.n_test, w.n_classes, w.n_cand)
    a, ref = _search_both(handle, w)
    for budget in (mn + (full - mn) // 3, mn):          # a few candidates per chunk; one candidate per chunk
        assert lb.workspace_bytes(arch, w.n_train, w.n_test, w.n_classes, w.n_cand, budget)[0] < full
        b, _ = _search_both(handle, w, budget=budget)
        for k in ("acc", "correct", "info", "best"):
            assert np.array_equal(a[k], b[k]), (k, budget)
        assert _fro(b["W_best"].astype(np.float64), a["W_best"].astype(np.float64)) <= 1e-6
    _check_search(handle, w, b, ref)


def test_auto_solver_flags_a_duplicated_kernel_and_fp64_recovers(handle):
    """Failure mode of the tensor-core Cholesky updates (LBCNN_SOLVER_AUTO from dimension 1024 on; ~2^-27 relative): a candidate
    whose LAST layer holds the same kernel twice has two identical feature maps, the system is singular up to the ridge, and
    the slice error may drive a pivot non-positive where the all-fp64 factorisation (and the oracle) succeeds.  Kernel sets
    are an input, so such a candidate can arrive.  What is required:
      - LBCNN_SOLVER_FP64: every candidate fits (info = 0) and matches the oracle;
      - LBCNN_SOLVER_AUTO: never silently wrong -- a candidate either matches the oracle or is flagged (info > 0, acc = -1,
        excluded from best / worst), and the healthy candidates are untouched by their neighbour's breakdown;
      - the documented recipe works: the flagged candidate re-run alone under LBCNN_SOLVER_FP64 fits and matches."""
    w = _small("gtsrb", 2600, 500, 3)
    trx, try_, tex, tey = synth.make_dataset(w)
    ker = synth.make_kernels(w).copy()
    l2 = 16 * 3 * 9                                   # layer 2 starts here; each of its kernels has 16 * 9 = 144 taps
    ker[1, l2 + 144:l2 + 288] = ker[1, l2:l2 + 144]   # candidate 1: layer-2 kernel 1 := kernel 0
    arch = lb.arch_of(w)
    args = lambda kk: (arch, _dev(trx), _dev(try_), _dev(tex), _dev(tey), w.n_classes, w.C, _dev(kk))
    ref = orc.search(_orc_arch(w), trx, try_, tex, tey, w.n_classes, w.C, ker, feature_scale=w.feature_scale, keep=True)
    assert (ref["info"] == 0).all()
    handle.set_workspace(None)
    handle.ensure_workspace(lb.workspace_bytes(arch, w.n_train, w.n_test, w.n_classes, w.n_cand)[0])
    try:
        handle.set_option(lb.OPT_SOLVER, lb.SOLVER_FP64)
        f = {k: v.cpu().numpy() for k, v in handle.search_candidates(*args(ker)).items()}
        assert (f["info"] == 0).all()
        assert (np.abs(f["acc"].astype(np.float64) - ref["acc"]) * 100.0 <= TOL_ACC_PP).all()
        handle.set_option(lb.OPT_SOLVER, lb.SOLVER_AUTO)
        a = {k: v.cpu().numpy() for k, v in handle.search_candidates(*args(ker)).items()}
        for k in range(w.n_cand):
            if a["info"][k] == 0:
                assert abs(float(a["acc"][k]) - ref["acc"][k]) * 100.0 <= TOL_ACC_PP, k
            else:
                assert k == 1 and a["info"][k] > 0 and a["acc"][k] == -1.0, (k, a["info"][k])
        assert a["info"][0] == 0 and a["info"][2] == 0
        assert int(a["best"][0]) != 1 or a["info"][1] == 0
        if a["info"][1] != 0:                          # the recipe of include/lbcnn.h: re-run what was flagged in fp64
            handle.set_option(lb.OPT_SOLVER, lb.SOLVER_FP64)
            r = {k: v.cpu().numpy() for k, v in handle.search_candidates(*args(ker[1:2])).items()}
            assert r["info"][0] == 0 and abs(float(r["acc"][0]) - ref["acc"][1]) * 100.0 <= TOL_ACC_PP
        print("AUTO info on the duplicated-kernel candidate:", int(a["info"][1]))
    finally:
        handle.set_option(lb.OPT_SOLVER, lb.SOLVER_AUTO)
        handle.set_workspace(None)


def test_search_chunked_equals_unchunked(handle):
    w = _small("mnist", 400, 150, 7)
    arch = lb.arch_of(w)
    full, mn = lb.workspace_bytes(arch, w.n_train, w.n_test, w.n_classes, w.n_cand)
    a, _ = _search_both(handle, w)
    # a workspace that only fits 2-3 candidates per chunk must give identical results
    b, _ = _search_both(handle, w, budget=mn + (full - mn) // 3)
    for k in ("acc", "correct", "info", "best", "W_best"):
        assert np.array_equal(a[k], b[k]), k
    handle.set_workspace(None)
    handle.ensure_workspace(mn - 256)
    trx, try_, tex, tey = synth.make_dataset(w)
    with pytest.raises(lb.LbcnnError) as e:
        handle.search_candidates(arch, _dev(trx), _dev(try_), _dev(tex), _dev(tey), w.n_classes, w.C,
                                 _dev(synth.make_kernels(w)))
    assert e.value.status == lb.ERR_WORKSPACE


def test_search_degenerate_sizes(handle):
    """one candidate (best = worst = 0), a single test sample (accuracy 0 or 1), a single train image
    per class-less corner: one image through the expander."""
    w = _small("mnist", 300, 1, 1)
    got, ref = _search_both(handle, w)
    assert int(got["best"][0]) == 0 and int(got["best"][1]) == 0
    assert got["acc"][0] in (0.0, 1.0) and got["acc"][0] == ref["acc"][0]
    assert _fro(got["W_best"].astype(np.float64), ref["W"][0]) <= TOL_W_FRO
    # one image, one candidate: every CTA of the tensor-core expander is a ragged batch
    w1 = _small("gtsrb", 50, 4, 1)
    x = synth.make_dataset(w1)[0][:1]
    ker = synth.make_kernels(w1, 1)
    H = handle.expand(lb.arch_of(w1, 1.0), _dev(x), _dev(ker)).cpu().numpy()
    assert np.array_equal(H[0].astype(np.int64), orc.expand(_orc_arch(w1), x, ker[0]))


def test_argument_errors_on_the_device_path(handle):
    w = _small("tiny_mnist", 64, 16, 2)
    trx, try_, tex, tey = synth.make_dataset(w)
    ker = synth.make_kernels(w)
    arch = lb.arch_of(w)
    handle.set_workspace(None)
    with pytest.raises(lb.LbcnnError) as e:          # no workspace at all
        handle.search_candidates(arch, _dev(trx), _dev(try_), _dev(tex), _dev(tey), w.n_classes, w.C, _dev(ker))
    assert e.value.status == lb.ERR_WORKSPACE
    handle.ensure_workspace(lb.workspace_bytes(arch, w.n_train, w.n_test, w.n_classes, w.n_cand)[0])
    for bad_C in (0.0, -1.0):                        # C <= 0
        with pytest.raises(lb.LbcnnError) as e:
            handle.search_candidates(arch, _dev(trx), _dev(try_), _dev(tex), _dev(tey), w.n_classes, bad_C, _dev(ker))
        assert e.value.status == lb.ERR_INVALID_ARG
    with pytest.raises(lb.LbcnnError) as e:          # fewer than two classes
        handle.search_candidates(arch, _dev(trx), _dev(try_), _dev(tex), _dev(tey), 1, w.C, _dev(ker))
    assert e.value.status == lb.ERR_INVALID_ARG
    bad = lb.make_arch(8, 8, 1, [(lb.CONV_FULL, 4, 4, 0, 2, 2, 0, 0)], 1.0)      # even kernel size
    with pytest.raises(lb.LbcnnError) as e:
        handle.expand(bad, _dev(trx[:, :8, :8]), _dev(ker))
    assert e.value.status == lb.ERR_INVALID_ARCH


def test_host_buffer_entry_equals_device_entry(handle):
    """lbcnn_search_candidates_host (bench.py's e2e leg) = the device-pointer entry on the same bytes."""
    w = _small("mnist", 500, 200, 6)
    trx, try_, tex, tey = synth.make_dataset(w)
    ker = synth.make_kernels(w)
    arch = lb.arch_of(w)
    full, _ = lb.workspace_bytes(arch, w.n_train, w.n_test, w.n_classes, w.n_cand)
    handle.set_workspace(None)
    handle.ensure_workspace(full + lb.host_staging_bytes(arch, w.n_train, w.n_test, w.n_classes, w.n_cand))
    dev = handle.search_candidates(arch, _dev(trx), _dev(try_), _dev(tex), _dev(tey), w.n_classes, w.C, _dev(ker))
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a))
    host = handle.search_candidates_host(arch, t(trx), t(try_), t(tex), t(tey), w.n_classes, w.C, t(ker))
    for k in ("acc", "correct", "info", "best", "W_best"):
        assert np.array_equal(dev[k].cpu().numpy(), host[k].numpy()), k


def test_staged_calls_replay_the_search(handle):
    """expand -> fit -> score through the three stand-alone entry points reproduces the driver's numbers
    (replay of the best kernels, PAPER.md:94 `use_stored`), and labels agree with the oracle's one by one."""
    w = _small("gtsrb", 1200, 400, 2)
    trx, try_, tex, tey = synth.make_dataset(w)
    ker = synth.make_kernels(w)
    got, ref = _search_both(handle, w)
    a1 = lb.arch_of(w, 1.0)
    Htr = handle.expand(a1, _dev(trx), _dev(ker))
    Hte = handle.expand(a1, _dev(tex), _dev(ker))
    s = float(np.float32(w.feature_scale))
    handle.set_workspace(None)
    handle.ensure_workspace(lb.workspace_bytes(a1, w.n_train, w.n_test, w.n_classes, w.n_cand)[0])
    W, info = handle.elm_fit(Htr, _dev(try_), w.n_classes, w.C, h_scale=s, flags=lb.H_INTEGER)
    pred, corr = handle.elm_score(Hte, W, _dev(tey), h_scale=s)
    assert np.array_equal(corr.cpu().numpy(), got["correct"])
    pred = pred.cpu().numpy()
    for k in range(w.n_cand):
        assert (pred[k] == ref["pred"][k]).mean() >= TOL_LABEL_AGREE
        assert _fro(W[k].cpu().numpy().astype(np.float64), ref["W"][k]) <= TOL_W_FRO


def test_full_size_bench_config_sampled(handle):
    """BASELINE configs[1] (the bench workload) at full size, in the launch configuration bench.py times:
    sampled feature rows, and two whole candidates' W / labels / accuracy, against the oracle."""
    w = synth.WORKLOADS["mnist"]
    trx, try_, tex, tey = synth.make_dataset(w)
    ker = synth.make_kernels(w)
    arch = lb.arch_of(w)
    full, _ = lb.workspace_bytes(arch, w.n_train, w.n_test, w.n_classes, w.n_cand)
    handle.set_workspace(None)
    handle.ensure_workspace(full)
    out = handle.search_candidates(arch, _dev(trx), _dev(try_), _dev(tex), _dev(tey), w.n_classes, w.C, _dev(ker))
    acc = out["acc"].cpu().numpy()
    correct = out["correct"].cpu().numpy()
    assert (out["info"].cpu().numpy() == 0).all()
    best = int(out["best"][0])
    assert best == int(np.argmax(correct)) and int(out["best"][1]) == int(np.argmin(correct))
    oa = _orc_arch(w)
    s = float(np.float32(w.feature_scale))
    # sampled feature rows of sampled candidates, through lbcnn_expand at full n
    rows = np.array([0, 1, 63, 64, 4097, 19999])
    H = handle.expand(lb.arch_of(w, 1.0), _dev(trx), _dev(ker[60:64])).cpu().numpy()
    for j, k in enumerate(range(60, 64)):
        assert np.array_equal(H[j][rows].astype(np.int64), orc.expand(oa, trx[rows], ker[k]))
    del H
    # the best candidate and candidate 0, whole: W, labels ONE BY ONE, accuracy
    cands = sorted({best, 0})
    ref_W, ref_pred = {}, {}
    for k in cands:
        Htr = orc.expand(oa, trx, ker[k]).astype(np.float64) * s
        Hte = orc.expand(oa, tex, ker[k]).astype(np.float64) * s
        Wo, inf, _ = orc.elm_fit(Htr, try_, w.n_classes, w.C)
        po, co, _ = orc.elm_score(Hte, Wo, tey)
        assert inf == 0
        ref_W[k], ref_pred[k] = Wo, po
        assert abs(co / w.n_test - acc[k]) * 100.0 <= TOL_ACC_PP
    assert _fro(out["W_best"].cpu().numpy().astype(np.float64), ref_W[best]) <= TOL_W_FRO
    del out
    _check_labels_and_W(handle, w, correct, ref_W, ref_pred, cands, data=(trx, try_, tex, tey))


def test_full_size_orl_config_sampled(handle):
    """BASELINE.json configs[3] at FULL size (1024 candidates, dual branch, 120 test samples: a single flipped label
    would break the 99.9 % / 0.2 pp tolerances) in the launch configuration bench.py times; eight candidates spread over
    the batch, the best and the worst are checked whole against the oracle -- every predicted label count must be equal."""
    w = synth.WORKLOADS["orl"]
    trx, try_, tex, tey = synth.make_dataset(w)
    ker = synth.make_kernels(w)
    arch = lb.arch_of(w)
    full, _ = lb.workspace_bytes(arch, w.n_train, w.n_test, w.n_classes, w.n_cand, int(100 * (1 << 30)))
    handle.set_workspace(None)
    handle.ensure_workspace(full)
    out = handle.search_candidates(arch, _dev(trx), _dev(try_), _dev(tex), _dev(tey), w.n_classes, w.C, _dev(ker))
    correct = out["correct"].cpu().numpy()
    acc = out["acc"].cpu().numpy()
    assert (out["info"].cpu().numpy() == 0).all()
    best, worst = int(out["best"][0]), int(out["best"][1])
    assert best == int(np.argmax(correct)) and worst == int(np.argmin(correct))
    oa = _orc_arch(w)
    s = float(np.float32(w.feature_scale))
    cands = sorted({0, 1, 127, 128, 511, 777, 1023, best, worst})
    ref_W, ref_pred = {}, {}
    for k in cands:
        Htr = orc.expand(oa, trx, ker[k]).astype(np.float64) * s
        Hte = orc.expand(oa, tex, ker[k]).astype(np.float64) * s
        Wo, inf, _ = orc.elm_fit(Htr, try_, w.n_classes, w.C)
        po, co, _ = orc.elm_score(Hte, Wo, tey)
        assert inf == 0
        ref_W[k], ref_pred[k] = Wo, po
        assert co == int(correct[k]), (k, co, int(correct[k]))
        assert abs(co / w.n_test - acc[k]) * 100.0 <= TOL_ACC_PP
    assert _fro(out["W_best"].cpu().numpy().astype(np.float64), ref_W[best]) <= TOL_W_FRO
    del out
    handle.set_workspace(None)
    # every predicted label (120 per candidate) and every W of the nine candidates
    _check_labels_and_W(handle, w, correct, ref_W, ref_pred, cands, data=(trx, try_, tex, tey))
    handle.set_workspace(None)


@pytest.mark.parametrize("name", ["gtsrb", "vggface"])
def test_full_size_expand_sampled(handle, name):
    """configs[2] / configs[4]: the expander at the FULL train-set size (the grid, batch and candidate split bench.py
    times); sampled rows -- first, last, around CTA batch boundaries -- of two candidates must equal the oracle's integers."""
    w = synth.WORKLOADS[name]
    trx = synth.make_dataset(w)[0]
    K0 = w.n_cand - 2
    ker = synth.make_kernels(w)[K0:]
    H = handle.expand(lb.arch_of(w, 1.0), _dev(trx), _dev(ker))
    n = w.n_train
    rows = np.array([0, 1, 2, 3, 5, 6, 7, n // 2, n // 2 + 1, n - 2, n - 1])
    Hs = H[:, torch.from_numpy(rows).cuda()].cpu().numpy()
    del H
    oa = _orc_arch(w)
    for j in range(2):
        assert np.array_equal(Hs[j].astype(np.int64), orc.expand(oa, trx[rows], ker[j])), (name, j)


def _fullsize_reference(name, w, trx, try_, tex, tey, ker, k, want_W=True):
    """the oracle's W / labels / margins of candidate k at full size: from tests/golden/fullsize_<name>.npz (written by
    tests/golden/make_fullsize_golden.py, which calls only oracle/) when its input key matches the bytes generated
    here, otherwise computed now by the oracle (minutes)."""
    import importlib.util
    import os
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    spec = importlib.util.spec_from_file_location("make_fullsize_golden", os.path.join(here, "make_fullsize_golden.py"))
    mk = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mk)
    key = mk.input_key(trx, try_, tex, tey, ker[k], w.C, float(np.float32(w.feature_scale)))
    path = mk.path_of(name)
    if os.path.exists(path):
        z = np.load(path)
        if ("key_%d" % k) in z.files and np.array_equal(z["key_%d" % k], key) and (("W_%d" % k) in z.files or not want_W):
            Wz = z["W_%d" % k].astype(np.float64) if ("W_%d" % k) in z.files else None      # W is stored for candidate 0 only
            return Wz, z["pred_%d" % k].astype(np.int32), int(z["correct_%d" % k]), z["margin_%d" % k].astype(np.float64)
    W, pred, corr, margin, info = mk.oracle_candidate(w, trx, try_, tex, tey, ker[k])
    assert info == 0
    return W, pred, corr, margin


@pytest.mark.parametrize("name", ["gtsrb", "vggface"])
def test_full_size_fit_score(handle, name):
    """BASELINE.json configs[2] / configs[4] at FULL size: one whole candidate through lbcnn_expand -> lbcnn_elm_fit
    (primal branch, F = 2048 / 8192 < N = 30000 / 20000, LBCNN_H_INTEGER: the Gram closest to the int32 exactness
    limit and the 8192^2 Cholesky) -> lbcnn_elm_score with d_pred, against the oracle: W relative Frobenius error,
    labels ONE BY ONE, accuracy -- and the search driver's own count for that candidate must equal the staged one."""
    w = synth.WORKLOADS[name]
    data = synth.make_dataset(w)
    trx, try_, tex, tey = data
    ker = synth.make_kernels(w)
    k = 0
    Wo, po, co, margin = _fullsize_reference(name, w, trx, try_, tex, tey, ker, k)
    handle.set_workspace(None)
    # the stand-alone fit takes the all-fp64 factorisation by default; LBCNN_SOLVER_MIXED is what the driver uses for these
    # two architectures (tensor-core trailing updates): both against the oracle
    W64, _, _, info64 = _staged(handle, w, trx, try_, tex, tey, ker[k:k + 1])
    assert info64[0] == 0 and _fro(W64[0], Wo) <= 1e-6
    try:
        handle.set_option(lb.OPT_SOLVER, lb.SOLVER_MIXED)
        W, pred, corr, info = _staged(handle, w, trx, try_, tex, tey, ker[k:k + 1])
    finally:
        handle.set_option(lb.OPT_SOLVER, lb.SOLVER_AUTO)
    assert info[0] == 0
    err = _fro(W[0], Wo)
    assert err <= TOL_W_FRO and err <= 1e-4, err
    differ = np.nonzero(pred[0] != po)[0]
    assert 1.0 - len(differ) / float(w.n_test) >= TOL_LABEL_AGREE, (len(differ), margin[differ][:10])
    assert abs(int(corr[0]) - co) / float(w.n_test) * 100.0 <= TOL_ACC_PP
    assert co == int((po == tey).sum())
    # the driver (the launch configuration bench.py times, first two candidates) counts the same for candidate 0
    handle.set_workspace(None)
    w2 = synth.scaled(w, n_cand=2)
    arch = lb.arch_of(w2)
    handle.ensure_workspace(lb.workspace_bytes(arch, w.n_train, w.n_test, w.n_classes, 2)[0])
    out = handle.search_candidates(arch, _dev(trx), _dev(try_), _dev(tex), _dev(tey), w.n_classes, w.C, _dev(ker[:2]))
    assert int(out["correct"][0].item()) == int(corr[0]) and int(out["info"][0].item()) == 0
    handle.set_workspace(None)


@pytest.mark.parametrize("name", ["gtsrb", "vggface"])
def test_full_size_driver_at_full_candidate_count(handle, name):
    """BASELINE.json configs[2] / configs[4] exactly as bench.py launches them: ALL 128 / 32 candidates at full N in one
    lbcnn_search_candidates call with bench.py's 100 GB workspace budget (chunk planning at 75 / 61 GB, grid.z = the whole
    batch, the band-major Gram tile order across candidates).  The first, the middle and the last candidate against the
    oracle's stored full-size result (tests/golden/fullsize_<name>.npz, written by the oracle-only script beside it):
    accuracy within 0.2 pp, and through the staged calls labels one by one; every candidate must fit (info = 0), the
    accuracies must follow from the counts, best / worst must be the first maximum / minimum of the counts."""
    import gc
    w = synth.WORKLOADS[name]
    data = synth.make_dataset(w)
    trx, try_, tex, tey = data
    ker = synth.make_kernels(w)
    K = w.n_cand
    arch = lb.arch_of(w)
    handle.set_workspace(None)
    gc.collect(); torch.cuda.empty_cache()
    handle.ensure_workspace(lb.workspace_bytes(arch, w.n_train, w.n_test, w.n_classes, K, 100 << 30)[0])
    out = handle.search_candidates(arch, _dev(trx), _dev(try_), _dev(tex), _dev(tey), w.n_classes, w.C, _dev(ker))
    torch.cuda.synchronize()
    got = {k: (v.cpu().numpy() if v is not None else None) for k, v in out.items()}
    handle.set_workspace(None)
    del out
    gc.collect(); torch.cuda.empty_cache()
    assert (got["info"] == 0).all()
    assert np.array_equal(got["acc"], (got["correct"].astype(np.float64) / w.n_test).astype(np.float32))
    assert int(got["best"][0]) == int(np.argmax(got["correct"])) and int(got["best"][1]) == int(np.argmin(got["correct"]))
    for k in (0, K // 2, K - 1):
        Wo, po, co, margin = _fullsize_reference(name, w, trx, try_, tex, tey, ker, k, want_W=(k == 0))
        assert co == int((po == tey).sum())
        assert abs(int(got["correct"][k]) - co) / float(w.n_test) * 100.0 <= TOL_ACC_PP, (k, int(got["correct"][k]), co)
        # labels one by one through the staged calls (same solver as the driver), tied to the driver by the equal count
        try:
            handle.set_option(lb.OPT_SOLVER, lb.SOLVER_MIXED)
            W, pred, corr, info = _staged(handle, w, trx, try_, tex, tey, ker[k:k + 1])
        finally:
            handle.set_option(lb.OPT_SOLVER, lb.SOLVER_AUTO)
        handle.set_workspace(None)
        assert info[0] == 0 and int(corr[0]) == int(got["correct"][k]), ("driver and staged calls disagree", k)
        differ = np.nonzero(pred[0] != po)[0]
        assert 1.0 - len(differ) / float(w.n_test) >= TOL_LABEL_AGREE, (k, len(differ), margin[differ][:10])
        if Wo is not None:
            assert _fro(W[0], Wo) <= 1e-4
            if int(got["best"][0]) == k:
                assert _fro(got["W_best"].astype(np.float64), Wo) <= TOL_W_FRO


# ---- exact integer Gram on the tensor cores (gram_tc.cu) -------------------------------------------------
TC_CASES = [  # n, F, c, max_abs, K : digits 1 / 2 / 3, ragged n (not a multiple of 64) and F (not of 16 / 96 / 128)
    (300, 70, 5, 100, 2), (1000, 200, 7, 30000, 3), (777, 333, 4, 900000, 2), (2049, 129, 3, 8000000, 1),
    (130, 97, 3, 20000, 2), (5000, 980, 10, 16000, 1),
    # F a multiple of 128: the label columns take an extra row of tiles
    (640, 256, 5, 20000, 2),
    # more than 128 classes: the right-hand side is NOT fused (label-segmented column sums)
    (700, 200, 130, 20000, 2),
    # dual branch (F >= n): K-major operands, contraction over the features; ragged n and F, 1 / 2 / 3 digits
    (150, 700, 5, 6000, 3), (97, 130, 3, 100, 2), (280, 5152, 40, 6375, 2), (200, 333, 4, 900000, 1)]


@pytest.mark.parametrize("n,F,c,amax,K", TC_CASES)
def test_integer_fit_tensor_core_gram_is_exact(handle, n, F, c, amax, K):
    """LBCNN_H_INTEGER routes the Gram through tcgen05 int8 digit planes; it must reproduce the fp64 SIMT
    Gram (flags = 0) exactly -- both are exact for integer data -- and the oracle's W within tolerance."""
    rng = np.random.default_rng(n * 131 + F)
    # low-rank + noise integer features with a common mode (ill-conditioned like the expander's output)
    base = rng.integers(-amax // 4, amax // 4, size=(K, 1, F))
    H = (base + rng.integers(-amax // 2, amax // 2, size=(K, n, F))).astype(np.float32)
    H[0, 0, 0] = float(amax - 1)
    H[0, 1, min(1, F - 1)] = float(-(amax - 1))
    y = rng.integers(0, c, size=n).astype(np.int32)
    s, Creg = 1.0 / 255.0, 1e3
    Hd, yd = _dev(H), _dev(y)
    handle.set_workspace(None)
    handle.ensure_workspace(64 << 20 if n * F < 3e5 else 1 << 30)
    W_tc, info_tc = handle.elm_fit(Hd, yd, c, Creg, h_scale=s, flags=lb.H_INTEGER)
    W_ref, info_ref = handle.elm_fit(Hd, yd, c, Creg, h_scale=s, flags=0)
    torch.cuda.synchronize()
    assert (info_tc.cpu().numpy() == 0).all() and (info_ref.cpu().numpy() == 0).all()
    assert torch.equal(W_tc, W_ref)
    sc = float(np.float32(s))
    Wo, inf, _ = orc.elm_fit(H[0].astype(np.float64) * sc, y, c, Creg)
    assert inf == 0 and _fro(W_tc[0].cpu().numpy().astype(np.float64), Wo) <= TOL_W_FRO
