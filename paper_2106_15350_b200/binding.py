"""Thin Python binding of liblbcnn.so (include/lbcnn.h): argument marshalling only.

Every step of the path runs in the CUDA library; torch supplies device memory and the current stream.
There is no CPU fallback: a missing library raises at import of the symbols, and a missing CUDA device
makes ``Handle()`` raise ``LbcnnError(LBCNN_ERR_CUDA)``.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence, Tuple

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "liblbcnn.so")

OK, ERR_INVALID_ARG, ERR_INVALID_ARCH, ERR_SHAPE, ERR_WORKSPACE, ERR_CUDA, ERR_NOMEM, ERR_STATIC_LIMIT = range(8)
EVOLVE_STATIC_MAX_CAND = 16384
CONV_FULL, CONV_DEPTHWISE = 0, 1
ACT_NONE, ACT_RELU = 0, 1
H_INTEGER, FORCE_PRIMAL, FORCE_DUAL = 1, 2, 4
EXPAND_SIMT, EXPAND_TENSOR = 0, 1
OPT_FORCE_SIMT_EXPAND, OPT_SOLVER, OPT_PANEL, OPT_DEFLATE, OPT_SCORER, OPT_MID_PANEL, OPT_STREAM_ROWS, OPT_DUAL_TRICK = 0, 1, 3, 5, 6, 7, 8, 9
SCORER_AUTO, SCORER_FP64, SCORER_TENSOR = 0, 1, 2
SOLVER_AUTO, SOLVER_FP64, SOLVER_MIXED = 0, 1, 2

EXPORTS = ("lbcnn_version", "lbcnn_status_string", "lbcnn_create", "lbcnn_destroy", "lbcnn_feature_dim",
           "lbcnn_kernel_set_size", "lbcnn_workspace_bytes", "lbcnn_set_workspace", "lbcnn_expand", "lbcnn_elm_fit",
           "lbcnn_elm_score", "lbcnn_search_candidates", "lbcnn_host_staging_bytes", "lbcnn_search_candidates_host",
           "lbcnn_launch_count", "lbcnn_set_profiling", "lbcnn_expand_path", "lbcnn_fit_workspace_bytes",
           "lbcnn_get_phase_times", "lbcnn_set_option", "lbcnn_expand_workspace_bytes", "lbcnn_get_op_stats", "lbcnn_score_workspace_bytes",
           "lbcnn_quantize_output_layer", "lbcnn_elm_score_q", "lbcnn_evolve_candidates", "lbcnn_evolve_candidates_static",
           "lbcnn_refine_workspace_bytes", "lbcnn_refine_output_layer")
PHASES = ("expand", "gram", "rhs", "solve", "score", "finish")


class Layer(C.Structure):
    _fields_ = [(n, C.c_int32) for n in
                ("conv_type", "n_kernels", "ksize", "act", "pool_k", "pool_s", "pool_p", "pool_cover_all")]


class Arch(C.Structure):
    _fields_ = [("in_h", C.c_int32), ("in_w", C.c_int32), ("in_c", C.c_int32), ("n_layers", C.c_int32),
                ("layer", Layer * 3), ("feature_scale", C.c_float)]


class RefineCfg(C.Structure):
    _fields_ = [("epochs", C.c_int32), ("batch", C.c_int32), ("lr", C.c_float), ("beta1", C.c_float), ("beta2", C.c_float),
                ("eps", C.c_float), ("seed", C.c_uint64)]


class LbcnnError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__("%s: status %d (%s)" % (where, status, status_string(status)))


_lib = None


def lib() -> C.CDLL:
    """Load liblbcnn.so (built in-tree by paper_2106_15350_b200.build).  Fails loudly when it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("liblbcnn.so is not built: run `python -m paper_2106_15350_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.lbcnn_version.restype = C.c_char_p
        L.lbcnn_status_string.restype = C.c_char_p
        L.lbcnn_status_string.argtypes = [C.c_int]
        for name in EXPORTS[2:]:
            getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def version() -> str:
    return lib().lbcnn_version().decode()


def status_string(status: int) -> str:
    return lib().lbcnn_status_string(int(status)).decode()


def _check(rc: int, where: str):
    if rc != OK:
        raise LbcnnError(rc, where)


def make_arch(in_h: int, in_w: int, in_c: int, layers: Sequence, feature_scale: float = 1.0) -> Arch:
    """layers: objects or tuples (conv_type, n_kernels, ksize, act, pool_k, pool_s, pool_p, pool_cover_all)."""
    a = Arch()
    a.in_h, a.in_w, a.in_c, a.n_layers = int(in_h), int(in_w), int(in_c), len(layers)
    a.feature_scale = float(feature_scale)
    if len(layers) > 3:
        raise LbcnnError(ERR_INVALID_ARCH, "make_arch")
    for i, L in enumerate(layers):
        t = tuple(L) if isinstance(L, (tuple, list)) else (
            L.conv_type, L.n_kernels, L.ksize, L.act, L.pool_k, L.pool_s, L.pool_p, L.pool_cover_all)
        for (name, _), v in zip(Layer._fields_, t):
            setattr(a.layer[i], name, int(v))
    return a


def arch_of(workload, feature_scale: Optional[float] = None) -> Arch:
    """Arch of a synth.Workload (plain data; synth.py holds no arithmetic of the method)."""
    fs = workload.feature_scale if feature_scale is None else feature_scale
    return make_arch(workload.in_h, workload.in_w, workload.in_c, workload.layers, fs)


def feature_dim(arch: Arch) -> Tuple[int, Tuple[int, int, int]]:
    F = C.c_int64()
    hwc = (C.c_int32 * 3)()
    _check(lib().lbcnn_feature_dim(C.byref(arch), C.byref(F), hwc), "lbcnn_feature_dim")
    return F.value, tuple(hwc)


def kernel_set_size(arch: Arch) -> Tuple[int, int]:
    nw, nb = C.c_int64(), C.c_int64()
    _check(lib().lbcnn_kernel_set_size(C.byref(arch), C.byref(nw), C.byref(nb)), "lbcnn_kernel_set_size")
    return nw.value, nb.value


def workspace_bytes(arch: Arch, n_train: int, n_test: int, n_classes: int, n_cand: int, budget_bytes: int = 0,
                    handle: "Optional[Handle]" = None) -> Tuple[int, int]:
    b, m = C.c_size_t(), C.c_size_t()
    h = handle._h if handle is not None else C.c_void_p(None)
    _check(lib().lbcnn_workspace_bytes(h, C.byref(arch), C.c_int64(n_train), C.c_int64(n_test), C.c_int32(n_classes),
                                       C.c_int32(n_cand), C.c_size_t(budget_bytes), C.byref(b), C.byref(m)),
           "lbcnn_workspace_bytes")
    return b.value, m.value


def fit_workspace_bytes(n: int, F: int, n_classes: int, n_cand: int, flags: int = 0) -> int:
    b = C.c_size_t()
    _check(lib().lbcnn_fit_workspace_bytes(C.c_int64(n), C.c_int64(F), C.c_int32(n_classes), C.c_int32(n_cand),
                                           C.c_uint32(flags), C.byref(b)), "lbcnn_fit_workspace_bytes")
    return b.value


def score_workspace_bytes(n: int, F: int, n_classes: int, n_cand: int) -> int:
    b = C.c_size_t()
    _check(lib().lbcnn_score_workspace_bytes(C.c_int64(n), C.c_int64(F), C.c_int32(n_classes), C.c_int32(n_cand), C.byref(b)),
           "lbcnn_score_workspace_bytes")
    return b.value


def host_staging_bytes(arch: Arch, n_train: int, n_test: int, n_classes: int, n_cand: int, has_bias: bool = False) -> int:
    b = C.c_size_t()
    _check(lib().lbcnn_host_staging_bytes(C.byref(arch), C.c_int64(n_train), C.c_int64(n_test), C.c_int32(n_classes),
                                          C.c_int32(n_cand), C.c_int32(int(has_bias)), C.byref(b)),
           "lbcnn_host_staging_bytes")
    return b.value


def _hptr(t, dtype=None, allow_none: bool = False):
    """host pointer of a contiguous CPU torch tensor (pinned or not) or NULL."""
    if t is None:
        if allow_none:
            return C.c_void_p(None)
        raise LbcnnError(ERR_INVALID_ARG, "null tensor")
    if t.is_cuda or not t.is_contiguous() or (dtype is not None and t.dtype != dtype):
        raise LbcnnError(ERR_INVALID_ARG, "tensor must be a contiguous CPU tensor of dtype %s" % dtype)
    return C.c_void_p(t.data_ptr())


def _ptr(t, dtype=None, allow_none: bool = False):
    """device pointer of a contiguous CUDA torch tensor (or NULL)."""
    if t is None:
        if allow_none:
            return C.c_void_p(None)
        raise LbcnnError(ERR_INVALID_ARG, "null tensor")
    if not t.is_cuda or not t.is_contiguous() or (dtype is not None and t.dtype != dtype):
        raise LbcnnError(ERR_INVALID_ARG, "tensor must be a contiguous CUDA tensor of dtype %s" % dtype)
    return C.c_void_p(t.data_ptr())


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


class Handle:
    """lbcnn_handle_t plus a caller-owned torch workspace buffer."""

    def __init__(self, device: int = 0):
        self._h = C.c_void_p(None)
        _check(lib().lbcnn_create(C.byref(self._h), int(device)), "lbcnn_create")
        self.device = int(device)
        self._ws = None

    def close(self):
        if self._h:
            lib().lbcnn_destroy(self._h)
            self._h = C.c_void_p(None)
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_workspace(self, ws):
        """ws: 1-D uint8 CUDA tensor (kept alive by the handle) or None."""
        if ws is None:
            _check(lib().lbcnn_set_workspace(self._h, C.c_void_p(None), C.c_size_t(0)), "lbcnn_set_workspace")
        else:
            _check(lib().lbcnn_set_workspace(self._h, _ptr(ws), C.c_size_t(ws.numel() * ws.element_size())),
                   "lbcnn_set_workspace")
        self._ws = ws

    def ensure_workspace(self, nbytes: int):
        import torch
        if self._ws is None or self._ws.numel() < nbytes:
            self._ws = None
            self.set_workspace(torch.empty(int(nbytes), dtype=torch.uint8, device="cuda:%d" % self.device))

    def set_option(self, option: int, value: int):
        _check(lib().lbcnn_set_option(self._h, C.c_int(option), C.c_int(value)), "lbcnn_set_option")

    def expand_workspace_bytes(self, arch: Arch, n_cand: int, has_bias: bool = False) -> int:
        b = C.c_size_t()
        _check(lib().lbcnn_expand_workspace_bytes(self._h, C.byref(arch), C.c_int32(n_cand), C.c_int32(int(has_bias)),
                                                  C.byref(b)), "lbcnn_expand_workspace_bytes")
        return b.value

    def expand_path(self, arch: Arch, has_bias: bool = False) -> int:
        """EXPAND_TENSOR (tcgen05 kernel) or EXPAND_SIMT (exact int32 kernel) for this architecture."""
        p = C.c_int32()
        _check(lib().lbcnn_expand_path(self._h, C.byref(arch), C.c_int32(int(has_bias)), C.byref(p)), "lbcnn_expand_path")
        return p.value

    def launch_count(self) -> int:
        n = C.c_int64()
        _check(lib().lbcnn_launch_count(self._h, C.byref(n)), "lbcnn_launch_count")
        return n.value

    def set_profiling(self, enable: bool):
        _check(lib().lbcnn_set_profiling(self._h, int(bool(enable))), "lbcnn_set_profiling")

    def phase_times(self):
        """blocks until the recorded phase events completed; returns {phase: (ms, brackets)}."""
        ms = (C.c_float * len(PHASES))()
        cnt = (C.c_int32 * len(PHASES))()
        _check(lib().lbcnn_get_phase_times(self._h, ms, cnt), "lbcnn_get_phase_times")
        return {p: (float(ms[i]), int(cnt[i])) for i, p in enumerate(PHASES)}

    def op_stats(self):
        """int8 multiply-adds (in units of 1e12) the tensor-core Gram / Cholesky trailing updates issued since the last
        call; synchronises and resets the device counters."""
        cnt = (C.c_uint64 * 2)()
        _check(lib().lbcnn_get_op_stats(self._h, cnt), "lbcnn_get_op_stats")
        return {"gram_int8_tmac": cnt[0] / 1e12, "solve_int8_tmac": cnt[1] / 1e12}

    # ---- the four calls of the path ----------------------------------------------------------
    def expand(self, arch: Arch, images, kernels, bias=None, out=None):
        """images u8 [n][H][W][C]; kernels i8 [K][n_weights]; returns H f32 [K][n][F]."""
        import torch
        F, _ = feature_dim(arch)
        n, K = images.shape[0], kernels.shape[0]
        if out is None:
            out = torch.empty((K, n, F), dtype=torch.float32, device=images.device)
        need = self.expand_workspace_bytes(arch, K, bias is not None)
        if need:
            self.ensure_workspace(need)
        _check(lib().lbcnn_expand(self._h, C.byref(arch), _ptr(images, torch.uint8), C.c_int64(n),
                                  _ptr(kernels, torch.int8), _ptr(bias, torch.int32, True), C.c_int32(K),
                                  _ptr(out, torch.float32), _stream()), "lbcnn_expand")
        return out

    def elm_fit(self, H, labels, n_classes: int, Creg: float, h_scale: float = 1.0, flags: int = 0):
        """H f32 [K][n][F]; returns (W f32 [K][F][c], info i32 [K])."""
        import torch
        K, n, F = H.shape
        W = torch.empty((K, F, n_classes), dtype=torch.float32, device=H.device)
        info = torch.empty((K,), dtype=torch.int32, device=H.device)
        _check(lib().lbcnn_elm_fit(self._h, _ptr(H, torch.float32), C.c_int64(n), C.c_int64(F), C.c_float(h_scale),
                                   C.c_uint32(flags), _ptr(labels, torch.int32), C.c_int32(n_classes), C.c_float(Creg),
                                   C.c_int32(K), _ptr(W), _ptr(info), _stream()), "lbcnn_elm_fit")
        return W, info

    def elm_score(self, H, W, labels=None, h_scale: float = 1.0, want_pred: bool = True):
        """returns (pred i32 [K][n] or None, correct i32 [K] or None)."""
        import torch
        K, n, F = H.shape
        c = W.shape[2]
        pred = torch.empty((K, n), dtype=torch.int32, device=H.device) if want_pred else None
        corr = torch.empty((K,), dtype=torch.int32, device=H.device) if labels is not None else None
        _check(lib().lbcnn_elm_score(self._h, _ptr(H, torch.float32), C.c_int64(n), C.c_int64(F), C.c_float(h_scale),
                                     _ptr(W, torch.float32), C.c_int32(c), _ptr(labels, torch.int32, True), C.c_int32(K),
                                     _ptr(pred, None, True), _ptr(corr, None, True), _stream()), "lbcnn_elm_score")
        return pred, corr

    def evolve_candidates(self, kernels, acc, n_elite: int, mut_ppm: int, seed: int, generation: int):
        """one generation of the genetic candidate generator: kernels i8 [K][n_weights], acc f32 [K] -> next i8 [K][n_weights]."""
        import torch
        K, nw = kernels.shape
        nxt = torch.empty_like(kernels)
        self.ensure_workspace(256 + 8 * K)
        _check(lib().lbcnn_evolve_candidates(self._h, _ptr(kernels, torch.int8), _ptr(acc, torch.float32), C.c_int32(K),
                                             C.c_int64(nw), C.c_int32(n_elite), C.c_uint32(mut_ppm), C.c_uint64(seed),
                                             C.c_uint32(generation), _ptr(nxt), _stream()), "lbcnn_evolve_candidates")
        return nxt

    def evolve_candidates_static(self, kernels, acc, n_elite: int, mut_ppm: int, seed: int, generation: int):
        """evolve_candidates for a caller that cannot allocate a workspace (a plug-in given only its input and output
        buffers, a process whose device memory is all spoken for, a loop that must not hit cudaMalloc's device-wide
        synchronisation): same arguments and byte-for-byte the same result, but the 8 bytes of ranking scratch per
        candidate come from a 128 KB array built into liblbcnn.so, so no workspace is set or needed and the C call
        allocates nothing.  (This Python wrapper still creates the output tensor, as evolve_candidates does; a caller that
        must not allocate goes through the C ABI with its own d_next.)  At most EVOLVE_STATIC_MAX_CAND candidates, else
        LbcnnError(ERR_STATIC_LIMIT).  The first call on a device resolves the array's address and may load the library's
        code there: make it at start-up, before any stream capture.  All handles and streams of a GPU share the one
        array, so calls that can overlap on the GPU race; keep them on one stream."""
        import torch
        K, nw = kernels.shape
        nxt = torch.empty_like(kernels)
        _check(lib().lbcnn_evolve_candidates_static(self._h, _ptr(kernels, torch.int8), _ptr(acc, torch.float32), C.c_int32(K),
                                                    C.c_int64(nw), C.c_int32(n_elite), C.c_uint32(mut_ppm), C.c_uint64(seed),
                                                    C.c_uint32(generation), _ptr(nxt), _stream()),
               "lbcnn_evolve_candidates_static")
        return nxt

    def refine_output_layer(self, H, labels, W, epochs: int = 10, batch: int = 128, lr: float = 1e-3, beta1: float = 0.9,
                            beta2: float = 0.999, eps: float = 1e-8, seed: int = 0, h_scale: float = 1.0):
        """H f32 [n][F], W f32 [F][c] (starting point; a refined copy is returned together with the per-epoch mean loss)."""
        import torch
        n, F = H.shape
        c = W.shape[1]
        cfg = RefineCfg(int(epochs), int(batch), float(lr), float(beta1), float(beta2), float(eps), int(seed))
        b = C.c_size_t()
        _check(lib().lbcnn_refine_workspace_bytes(C.c_int64(F), C.c_int32(c), C.byref(cfg), C.byref(b)), "lbcnn_refine_workspace_bytes")
        self.ensure_workspace(b.value)
        Wn = W.clone()
        loss = torch.zeros(max(int(epochs), 1), dtype=torch.float32, device=H.device)
        _check(lib().lbcnn_refine_output_layer(self._h, _ptr(H, torch.float32), C.c_int64(n), C.c_int64(F), C.c_float(h_scale),
                                               _ptr(labels, torch.int32), C.c_int32(c), C.byref(cfg), _ptr(Wn, torch.float32),
                                               _ptr(loss), _stream()), "lbcnn_refine_output_layer")
        return Wn, loss[:int(epochs)]

    def quantize_output_layer(self, W, bits: int = 8):
        """W f32 [K][F][c] -> (Wq i8 [K][F][c], scale f32 [K]); W ~ scale * Wq (include/lbcnn.h)."""
        import torch
        K, F, c = W.shape
        Wq = torch.empty((K, F, c), dtype=torch.int8, device=W.device)
        scale = torch.empty((K,), dtype=torch.float32, device=W.device)
        _check(lib().lbcnn_quantize_output_layer(self._h, _ptr(W, torch.float32), C.c_int64(F), C.c_int32(c), C.c_int32(K),
                                                 C.c_int32(bits), _ptr(Wq), _ptr(scale), _stream()), "lbcnn_quantize_output_layer")
        return Wq, scale

    def elm_score_q(self, H, Wq, labels=None, want_pred: bool = True):
        """returns (pred i32 [K][n] or None, correct i32 [K] or None) with the int8 output layer."""
        import torch
        K, n, F = H.shape
        c = Wq.shape[2]
        self.ensure_workspace(score_workspace_bytes(n, F, c, K))
        pred = torch.empty((K, n), dtype=torch.int32, device=H.device) if want_pred else None
        corr = torch.empty((K,), dtype=torch.int32, device=H.device) if labels is not None else None
        _check(lib().lbcnn_elm_score_q(self._h, _ptr(H, torch.float32), C.c_int64(n), C.c_int64(F), _ptr(Wq, torch.int8),
                                       C.c_int32(c), _ptr(labels, torch.int32, True), C.c_int32(K), _ptr(pred, None, True),
                                       _ptr(corr, None, True), _stream()), "lbcnn_elm_score_q")
        return pred, corr

    def search_candidates(self, arch: Arch, train_x, train_y, test_x, test_y, n_classes: int, Creg: float, kernels,
                          bias=None, want_W: bool = True, out=None):
        """returns dict(acc f32 [K], correct i32 [K], info i32 [K], best i32 [2], W_best f32 [F][c] or None);
        everything stays on the device."""
        import torch
        F, _ = feature_dim(arch)
        K = kernels.shape[0]
        dev = train_x.device
        if out is None:
            out = dict(acc=torch.empty(K, dtype=torch.float32, device=dev),
                       correct=torch.empty(K, dtype=torch.int32, device=dev),
                       info=torch.empty(K, dtype=torch.int32, device=dev),
                       best=torch.empty(2, dtype=torch.int32, device=dev),
                       W_best=torch.empty((F, n_classes), dtype=torch.float32, device=dev) if want_W else None)
        _check(lib().lbcnn_search_candidates(
            self._h, C.byref(arch), _ptr(train_x, torch.uint8), _ptr(train_y, torch.int32), C.c_int64(train_x.shape[0]),
            _ptr(test_x, torch.uint8), _ptr(test_y, torch.int32), C.c_int64(test_x.shape[0]), C.c_int32(n_classes),
            C.c_float(Creg), _ptr(kernels, torch.int8), _ptr(bias, torch.int32, True), C.c_int32(K),
            _ptr(out["acc"]), _ptr(out["correct"]), _ptr(out["info"]), _ptr(out["best"]),
            _ptr(out["W_best"], None, True), _stream()), "lbcnn_search_candidates")
        return out

    def search_candidates_host(self, arch: Arch, train_x, train_y, test_x, test_y, n_classes: int, Creg: float,
                               kernels, bias=None, want_W: bool = True, out=None):
        """lbcnn_search_candidates_host: all tensors are CPU tensors (pin them for asynchronous copies); the
        call copies them in, runs the loop, copies the results back and synchronises.  Returns CPU tensors."""
        import torch
        F, _ = feature_dim(arch)
        K = kernels.shape[0]
        if out is None:
            pin = torch.cuda.is_available()
            out = dict(acc=torch.empty(K, dtype=torch.float32, pin_memory=pin),
                       correct=torch.empty(K, dtype=torch.int32, pin_memory=pin),
                       info=torch.empty(K, dtype=torch.int32, pin_memory=pin),
                       best=torch.empty(2, dtype=torch.int32, pin_memory=pin),
                       W_best=torch.empty((F, n_classes), dtype=torch.float32, pin_memory=pin) if want_W else None)
        _check(lib().lbcnn_search_candidates_host(
            self._h, C.byref(arch), _hptr(train_x, torch.uint8), _hptr(train_y, torch.int32),
            C.c_int64(train_x.shape[0]), _hptr(test_x, torch.uint8), _hptr(test_y, torch.int32),
            C.c_int64(test_x.shape[0]), C.c_int32(n_classes), C.c_float(Creg), _hptr(kernels, torch.int8),
            _hptr(bias, torch.int32, True), C.c_int32(K), _hptr(out["acc"]), _hptr(out["correct"]), _hptr(out["info"]),
            _hptr(out["best"]), _hptr(out["W_best"], None, True), _stream()), "lbcnn_search_candidates_host")
        return out
