"""C-ABI library: it builds, loads and exports every symbol include/lbcnn.h declares; the host-only
shape helpers agree with the paper's printed sizes.  No compute call is made here (no GPU needed)."""
import ctypes as C
import os
import re

import pytest

from paper_2106_15350_b200 import binding as lb
from paper_2106_15350_b200 import build as lbbuild
from paper_2106_15350_b200 import synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PAPER_POOL = (4, 2, 1, 1)


@pytest.fixture(scope="module", autouse=True)
def _built():
    lbbuild.build()


def _declared():
    text = open(os.path.join(ROOT, "include", "lbcnn.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lbcnn_[a-z_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported():
    names = _declared()
    assert set(names) == set(lb.EXPORTS), (names, lb.EXPORTS)
    L = lb.lib()
    for n in names:
        assert hasattr(L, n), n


def test_version_and_status_strings():
    assert "sm_100a" in lb.version()
    assert lb.status_string(0) == "ok"
    assert len({lb.status_string(i) for i in range(8)}) == 8
    assert "built-in scratch" in lb.status_string(lb.ERR_STATIC_LIMIT)      # lbcnn_evolve_candidates_static's size refusal
    assert lb.status_string(99) == "unknown status"


def _dw_arch(h, w, c, mult):
    return lb.make_arch(h, w, c, [(lb.CONV_DEPTHWISE, m, 3, 0) + PAPER_POOL for m in mult])


def test_feature_dim_paper_anchors():
    # MNIST 28x28x1, depthwise (16,20), pool 4/stride 2 -> F = 15680
    assert lb.feature_dim(_dw_arch(28, 28, 1, (16, 20))) == (15680, (7, 7, 320))
    # Table II (40,2,2): 204.8 kbit / 8 bit / 10 classes = 2560 = 4*4*160 (cover_all pinned) PAPER.md:140
    assert lb.feature_dim(_dw_arch(28, 28, 1, (40, 2, 2)))[0] == 2560
    # Table III GTSRB (13): 3434496 bit / 8 / 43 = 9984 PAPER.md:152
    assert lb.feature_dim(_dw_arch(32, 32, 3, (13,)))[0] == 9984
    # Table V VGG6 (20,4,4): 2949120 / 8 / 6 = 61440 PAPER.md:183
    assert lb.feature_dim(_dw_arch(64, 64, 3, (20, 4, 4)))[0] == 61440


@pytest.mark.parametrize("name,F", [("tiny_mnist", 196), ("mnist", 980), ("gtsrb", 2048), ("orl", 5152),
                                    ("vggface", 8192), ("paper_anchor", 15680)])
def test_feature_dim_and_kernel_set_size_of_configs(name, F):
    w = synth.WORKLOADS[name]
    a = lb.arch_of(w)
    assert lb.feature_dim(a)[0] == F
    assert lb.kernel_set_size(a) == synth.kernel_set_size(w)


def test_invalid_arch_status():
    with pytest.raises(lb.LbcnnError) as e:
        lb.feature_dim(lb.make_arch(28, 28, 1, [(0, 4, 4, 0, 2, 2, 0, 0)]))     # even kernel size
    assert e.value.status == lb.ERR_INVALID_ARCH
    with pytest.raises(lb.LbcnnError) as e:
        lb.feature_dim(lb.make_arch(2, 2, 1, [(0, 4, 3, 0, 4, 4, 0, 0)]))       # pooling window larger than the map
    assert e.value.status == lb.ERR_INVALID_ARCH
    with pytest.raises(lb.LbcnnError) as e:
        lb.feature_dim(lb.make_arch(8, 8, 1, []))
    assert e.value.status == lb.ERR_INVALID_ARCH


def test_workspace_bytes_is_host_arithmetic():
    w = synth.WORKLOADS["mnist"]
    a = lb.arch_of(w)
    full, mn = lb.workspace_bytes(a, w.n_train, w.n_test, w.n_classes, w.n_cand)
    assert mn < full
    # H for all candidates dominates: 64 * 30000 * 980 * 4 bytes
    assert full > 64 * 30000 * 980 * 4
    capped, _ = lb.workspace_bytes(a, w.n_train, w.n_test, w.n_classes, w.n_cand, budget_bytes=2 << 30)
    assert mn <= capped <= (2 << 30)
    with pytest.raises(lb.LbcnnError):
        lb.workspace_bytes(a, 0, 10, 10, 1)


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(lb.LbcnnError) as e:
        lb.Handle(0)
    assert e.value.status == lb.ERR_CUDA


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2106_15350_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", src, flags=re.M), f
                assert "liblbcnn_oracle" not in src, f
