// api.cu -- the C ABI of liblbcnn (include/lbcnn.h): argument checking, shape arithmetic, workspace
// planning and the search driver.  All compute is in expand.cu / fit.cu / score.cu; there is no CPU path.
#include "internal.h"
#include <new>

// ---- host shape logic -------------------------------------------------------------------------
// pooling output size (PAPER.md:54 max_pooling_2d(ksize, stride, pad, cover_all=True); PAPER.md:104 28->14->7)
int lb_pool_out(int n, int k, int s, int p, int cover_all) {
  if (n < 1 || k < 1 || s < 1 || p < 0) return -1;
  const int span = n + 2 * p - k;
  if (span < 0) return -1;
  const int out = (cover_all ? (span + s - 1) / s : span / s) + 1;
  // first and last windows must hold a real cell (windows in between then do as well when s <= k; check all)
  for (int i = 0; i < out; ++i) {
    int lo = i * s - p, hi = lo + k;
    if (lo < 0) lo = 0;
    if (hi > n) hi = n;
    if (hi <= lo) return -1;
  }
  return out;
}

int lb_arch_shape(const lbcnn_arch_t* a, ArchShape* s) {
  if (!a || !s) return LBCNN_ERR_INVALID_ARG;
  if (a->n_layers < 1 || a->n_layers > 3 || a->in_h < 1 || a->in_w < 1 || a->in_c < 1) return LBCNN_ERR_INVALID_ARCH;
  int h = a->in_h, w = a->in_w, c = a->in_c;
  int64_t w_off = 0, b_off = 0;
  long double bound = 255.0L;
  s->n_layers = a->n_layers;
  for (int l = 0; l < a->n_layers; ++l) {
    const lbcnn_layer_t& A = a->layer[l];
    LayerShape& L = s->L[l];
    if (A.n_kernels < 1 || A.ksize < 1 || (A.ksize % 2) == 0) return LBCNN_ERR_INVALID_ARCH;
    if (A.conv_type != LBCNN_CONV_FULL && A.conv_type != LBCNN_CONV_DEPTHWISE) return LBCNN_ERR_INVALID_ARCH;
    if (A.act != LBCNN_ACT_NONE && A.act != LBCNN_ACT_RELU) return LBCNN_ERR_INVALID_ARCH;
    L.conv_type = A.conv_type; L.nk = A.n_kernels; L.k = A.ksize; L.act = A.act;
    L.pk = A.pool_k; L.ps = A.pool_s; L.pp = A.pool_p; L.cover = A.pool_cover_all;
    L.cin = c; L.hin = h; L.win = w;
    L.cout = (A.conv_type == LBCNN_CONV_FULL) ? A.n_kernels : c * A.n_kernels;
    L.hout = lb_pool_out(h, A.pool_k, A.pool_s, A.pool_p, A.pool_cover_all);
    L.wout = lb_pool_out(w, A.pool_k, A.pool_s, A.pool_p, A.pool_cover_all);
    if (L.hout < 1 || L.wout < 1) return LBCNN_ERR_INVALID_ARCH;
    L.w_off = w_off; L.b_off = b_off;
    w_off += (int64_t)A.n_kernels * c * A.ksize * A.ksize;
    b_off += L.cout;
    bound *= (long double)A.ksize * A.ksize * (A.conv_type == LBCNN_CONV_FULL ? c : 1);
    h = L.hout; w = L.wout; c = L.cout;
  }
  s->F = (int64_t)c * h * w;
  s->n_weights = w_off; s->n_bias = b_off;
  s->max_abs = bound > 4.0e18L ? (int64_t)4000000000000000000LL : (int64_t)bound;
  return LBCNN_OK;
}

// ---- plain entry points -------------------------------------------------------------------------
extern "C" {

const char* lbcnn_version(void) { return "lbcnn-b200 0.1 (sm_100a)"; }

const char* lbcnn_status_string(int status) {
  switch (status) {
    case LBCNN_OK: return "ok";
    case LBCNN_ERR_INVALID_ARG: return "invalid argument";
    case LBCNN_ERR_INVALID_ARCH: return "invalid architecture";
    case LBCNN_ERR_SHAPE: return "shape mismatch";
    case LBCNN_ERR_WORKSPACE: return "workspace absent or too small";
    case LBCNN_ERR_CUDA: return "CUDA error (no device, launch or driver failure)";
    case LBCNN_ERR_NOMEM: return "host allocation failed";
    case LBCNN_ERR_STATIC_LIMIT: return "size beyond the capacity of the library's built-in scratch array (use the workspace variant)";
    default: return "unknown status";
  }
}

int lbcnn_create(lbcnn_handle_t* h, int device) {
  if (!h) return LBCNN_ERR_INVALID_ARG;
  *h = nullptr;
  int count = 0;
  if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) return LBCNN_ERR_CUDA;
  // the attributes are queried by device ordinal: the calling thread's current device is left as it was
  int n_sm = 0, smem_optin = 0;
  LB_CUDA_OK(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, device));
  LB_CUDA_OK(cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device));
  lbcnn_handle_s* p = new (std::nothrow) lbcnn_handle_s();
  if (!p) return LBCNN_ERR_NOMEM;
  p->device = device; p->n_sm = n_sm; p->max_smem_optin = smem_optin;
  p->ws = nullptr; p->ws_bytes = 0; p->launches = 0; p->profiling = 0;
  p->force_simt_expand = 0; p->solver = LBCNN_SOLVER_AUTO; p->panel = 1024; p->deflate = 16; p->dual_trick = 1; p->stream_rows = 0; p->mid_panel = 256; p->scorer = LBCNN_SCORER_AUTO;
  *h = p;
  return LBCNN_OK;
}

int lbcnn_set_option(lbcnn_handle_t h, int option, int value) {
  if (!h) return LBCNN_ERR_INVALID_ARG;
  switch (option) {
    case LBCNN_OPT_FORCE_SIMT_EXPAND: h->force_simt_expand = value ? 1 : 0; return LBCNN_OK;
    case LBCNN_OPT_SOLVER:
      if (value != LBCNN_SOLVER_AUTO && value != LBCNN_SOLVER_FP64 && value != LBCNN_SOLVER_MIXED) return LBCNN_ERR_INVALID_ARG;
      h->solver = value; return LBCNN_OK;
    case LBCNN_OPT_DEFLATE:
      if (value < 0 || value > 64) return LBCNN_ERR_INVALID_ARG;
      h->deflate = value; return LBCNN_OK;
    case LBCNN_OPT_SCORER:
      if (value != LBCNN_SCORER_AUTO && value != LBCNN_SCORER_FP64 && value != LBCNN_SCORER_TENSOR) return LBCNN_ERR_INVALID_ARG;
      h->scorer = value; return LBCNN_OK;
    case LBCNN_OPT_MID_PANEL:
      if (value != 0 && (value < 64 || value > LB_STC_KMAX || value % 64)) return LBCNN_ERR_INVALID_ARG;
      h->mid_panel = value; return LBCNN_OK;
    case LBCNN_OPT_STREAM_ROWS:
      if (value < 0) return LBCNN_ERR_INVALID_ARG;
      h->stream_rows = value; return LBCNN_OK;
    case LBCNN_OPT_DUAL_TRICK: h->dual_trick = value ? 1 : 0; return LBCNN_OK;
    case LBCNN_OPT_PANEL:
      if (value < 64 || value > LB_STC_KMAX || value % 64) return LBCNN_ERR_INVALID_ARG;
      h->panel = value; return LBCNN_OK;
    default: return LBCNN_ERR_INVALID_ARG;
  }
}

int lbcnn_set_profiling(lbcnn_handle_t h, int enable) {
  if (!h) return LBCNN_ERR_INVALID_ARG;
  h->profiling = enable ? 1 : 0;
  return LBCNN_OK;
}

int lbcnn_get_phase_times(lbcnn_handle_t h, float* h_ms, int32_t* h_count) {
  if (!h || !h_ms || !h_count) return LBCNN_ERR_INVALID_ARG;
  for (int i = 0; i < LBCNN_N_PHASES; ++i) { h_ms[i] = 0.0f; h_count[i] = 0; }
  int rc = LBCNN_OK;
  for (LbPhaseRec& r : h->recs) {
    float ms = 0.0f;
    if (cudaEventSynchronize(r.stop) != cudaSuccess || cudaEventElapsedTime(&ms, r.start, r.stop) != cudaSuccess)
      rc = LBCNN_ERR_CUDA;
    if (r.phase >= 0 && r.phase < LBCNN_N_PHASES) { h_ms[r.phase] += ms; h_count[r.phase] += 1; }
    cudaEventDestroy(r.start); cudaEventDestroy(r.stop);
  }
  h->recs.clear();
  return rc;
}

int lbcnn_destroy(lbcnn_handle_t h) {
  if (!h) return LBCNN_ERR_INVALID_ARG;
  for (LbPhaseRec& r : h->recs) { cudaEventDestroy(r.start); cudaEventDestroy(r.stop); }
  delete h;
  return LBCNN_OK;
}

int lbcnn_feature_dim(const lbcnn_arch_t* arch, int64_t* F, int32_t out_hwc[3]) {
  ArchShape s;
  const int rc = lb_arch_shape(arch, &s);
  if (rc) return rc;
  if (F) *F = s.F;
  if (out_hwc) {
    const LayerShape& L = s.L[s.n_layers - 1];
    out_hwc[0] = L.hout; out_hwc[1] = L.wout; out_hwc[2] = L.cout;
  }
  return LBCNN_OK;
}

int lbcnn_kernel_set_size(const lbcnn_arch_t* arch, int64_t* n_weights, int64_t* n_bias) {
  ArchShape s;
  const int rc = lb_arch_shape(arch, &s);
  if (rc) return rc;
  if (n_weights) *n_weights = s.n_weights;
  if (n_bias) *n_bias = s.n_bias;
  return LBCNN_OK;
}

int lbcnn_launch_count(lbcnn_handle_t h, int64_t* count) {
  if (!h || !count) return LBCNN_ERR_INVALID_ARG;
  *count = h->launches;
  return LBCNN_OK;
}

int lbcnn_set_workspace(lbcnn_handle_t h, void* d_ws, size_t bytes) {
  if (!h) return LBCNN_ERR_INVALID_ARG;
  if ((d_ws == nullptr) != (bytes == 0)) return LBCNN_ERR_INVALID_ARG;
  if (reinterpret_cast<uintptr_t>(d_ws) % 256 != 0) return LBCNN_ERR_INVALID_ARG;
  if (d_ws && bytes < LB_WS_HEAD) return LBCNN_ERR_INVALID_ARG;
  h->ws = d_ws; h->ws_bytes = bytes;
  if (d_ws) LB_CUDA_OK(cudaMemset(d_ws, 0, LB_WS_HEAD));     // the measurement counters at the head of the workspace (a configuration call: blocking)
  return LBCNN_OK;
}

int lbcnn_get_op_stats(lbcnn_handle_t h, uint64_t* h_counts) {
  if (!h || !h_counts) return LBCNN_ERR_INVALID_ARG;
  h_counts[0] = 0; h_counts[1] = 0;
  if (!h->ws) return LBCNN_OK;
  unsigned long long tmp[2] = {0ull, 0ull};
  LB_CUDA_OK(cudaMemcpy(tmp, h->ws, sizeof(tmp), cudaMemcpyDeviceToHost));      // synchronises: a measurement call
  LB_CUDA_OK(cudaMemset(h->ws, 0, sizeof(tmp)));
  h_counts[0] = tmp[0]; h_counts[1] = tmp[1];
  return LBCNN_OK;
}

}  // extern "C"

// ---- workspace planning for the search driver ---------------------------------------------------
namespace {
struct SearchPlan {
  FitPlan fit;
  size_t xw_off, fit_off, htr_off, hte_off, w_off, sc_off, gs_off, total;
  int stream; int64_t ntr_ws, nte_ws;      // streamed: rows of the train / test features resident at once
  int dual_kt;                             // dual branch scored through the kernel trick: train and test features stacked in one buffer
};
// xw1 = expander scratch per candidate (lb_expand_ws_bytes(.., 1)); kc = candidates per chunk
// sr: streamed search (LBCNN_OPT_STREAM_ROWS) -- at most sr samples of the train / test set are resident at once
// gs: bytes of one candidate's kernel set + bias (the slot a chunked kernel-trick search gathers its best candidate into)
void plan_search(int64_t F, int64_t n_train, int64_t n_test, int c, int n_cand, int kc, uint32_t flags, size_t xw1, int64_t sr,
                 size_t gs, SearchPlan* p, bool dual_kt = true) {
  // The streamed plan is judged on the chunk it would contract per launch, not on the whole set: N_train = 60000 is beyond
  // the exact Gram's int32 bound as one launch and inside it as chunks.  A request for longer chunks than that bound is
  // served with chunks of the bound ("at most r samples at a time" still holds).
  const int64_t sr_tr = (sr > LB_GRAM_TC_MAX_K) ? LB_GRAM_TC_MAX_K : sr;
  const bool chunk_train = sr_tr > 0 && sr_tr < n_train;
  lb_fit_plan(n_train, F, c, kc, flags, &p->fit, chunk_train ? sr_tr : 0);
  p->stream = (sr > 0 && (chunk_train || sr < n_test) && p->fit.primal && p->fit.use_tc && p->fit.fuse_rhs) ? 1 : 0;
  if (p->stream) {
    if (chunk_train) n_train = sr_tr;
    if (sr < n_test) n_test = sr;
  } else if (chunk_train) {
    lb_fit_plan(n_train, F, c, kc, flags, &p->fit);      // not streamable (dual branch, bias, > 128 classes, ...): the resident plan
  }
  p->ntr_ws = n_train; p->nte_ws = n_test;
  // dual branch with the exact tensor-core Gram: test rows are stacked behind the train rows, the Gram of the stack carries
  // the cross-Gram and the scores come out of the factorisation (fit.cu, DualScore).  Taken whatever the chunk size, so that
  // the decisions (correct[], acc, best) do not depend on how much workspace the caller gave.
  p->dual_kt = (dual_kt && !p->fit.primal && p->fit.use_tc) ? 1 : 0;
  if (p->dual_kt) lb_fit_plan(n_train, F, c, kc, flags, &p->fit, 0, n_test);
  size_t off = 0;
  p->xw_off = off;  off += (size_t)lb_align_up((int64_t)(xw1 * (size_t)kc), 256);
  p->fit_off = off; off += p->fit.total;
  p->htr_off = off; off += (size_t)lb_align_up((int64_t)kc * (n_train + (p->dual_kt ? n_test : 0)) * F * 4, 256);
  p->hte_off = off; off += p->dual_kt ? 0 : (size_t)lb_align_up((int64_t)kc * n_test * F * 4, 256);
  p->w_off = off;   off += (size_t)lb_align_up((int64_t)n_cand * F * c * 4, 256);
  // scratch of the tensor-core scorer (integer features only; it may still be left unused at run time)
  p->sc_off = off;  if (flags & LBCNN_H_INTEGER) off += lb_score_tc_ws_bytes(n_test, F, c, kc);
  // kernel-trick search in several chunks: slot for the best candidate's kernel set, bias and the info word of its re-fit
  p->gs_off = off;  if (p->dual_kt && kc < n_cand) off += (size_t)lb_align_up((int64_t)gs, 256) + 256;
  p->total = off;
}
// The driver's features are exact integers; inside the digit envelope of the exact tensor-core Gram (three balanced
// radix-256 digits hold |u| <= 8355711) the fit may use it.  A bias is an arbitrary int32 and is not part of the bound,
// so a search with bias keeps the general fp64 Gram.
// The tensor-core Cholesky updates carry ~2^-27 relative error: fine for the conditioning of distinct random features
// (cond ~1e6), fatal for a system that is singular up to the ridge -- two identical or negated feature maps.  That happens
// when two +-1 kernels of the LAST layer coincide: with t = Cin k^2 taps the chance per pair is 2^(1-t).  A depthwise last
// layer (t = k^2 = 9: about every second candidate of the paper's (16,20) architecture) or a tiny full one must keep the
// all-fp64 solver; from 32 taps on (configs[2], [4]: 144) the chance is below 1e-9 per pair.
bool arch_allows_tc_solver(const ArchShape& s) {
  const LayerShape& L = s.L[s.n_layers - 1];
  return L.conv_type == LBCNN_CONV_FULL && (int64_t)L.cin * L.k * L.k >= 32;
}

uint32_t search_fit_flags(const ArchShape& s, bool has_bias) {
  return (!has_bias && s.max_abs <= LB_H_INTEGER_MAX) ? LBCNN_H_INTEGER : 0u;
}
// largest chunk size whose plan fits in `bytes` (0 if none)
int fit_chunk(int64_t F, int64_t n_train, int64_t n_test, int c, int n_cand, uint32_t flags, size_t xw1, int64_t sr, size_t gs,
              size_t bytes, bool dual_kt = true) {
  SearchPlan p;
  plan_search(F, n_train, n_test, c, n_cand, n_cand, flags, xw1, sr, gs, &p, dual_kt);
  if (p.total <= bytes) return n_cand;
  int lo = 0, hi = n_cand;   // plan(lo) fits (lo = 0 means none), plan(hi) does not
  while (hi - lo > 1) {
    const int mid = lo + (hi - lo) / 2;
    plan_search(F, n_train, n_test, c, n_cand, mid, flags, xw1, sr, gs, &p, dual_kt);
    if (p.total <= bytes) lo = mid; else hi = mid;
  }
  return lo;
}
// expander scratch per candidate; a NULL handle (pure host arithmetic) assumes the B200's 227 KB of shared memory
size_t gather_slot_bytes(const ArchShape& s) { return (size_t)lb_align_up(s.n_weights, 256) + (size_t)s.n_bias * 4; }
size_t expand_ws_per_cand(lbcnn_handle_t h, const ArchShape& s, bool has_bias) {
  lbcnn_handle_s tmp{};
  tmp.max_smem_optin = 232448;
  return lb_expand_ws_bytes(h ? h : &tmp, s, has_bias, 1);
}
}  // namespace

extern "C" {

int lbcnn_workspace_bytes(lbcnn_handle_t h, const lbcnn_arch_t* arch, int64_t n_train, int64_t n_test,
                          int32_t n_classes, int32_t n_cand, size_t budget_bytes, size_t* bytes, size_t* min_bytes) {
  if (!bytes || n_train < 1 || n_test < 0 || n_classes < 2 || n_cand < 1) return LBCNN_ERR_INVALID_ARG;
  ArchShape s;
  const int rc = lb_arch_shape(arch, &s);
  if (rc) return rc;
  const uint32_t flags = search_fit_flags(s, false);     // the bias-free plan is the larger one (digit planes)
  const size_t xw1 = expand_ws_per_cand(h, s, false);
  const int64_t sr = h ? h->stream_rows : 0;
  const size_t gs = gather_slot_bytes(s);
  SearchPlan p1, p1n;
  plan_search(s.F, n_train, n_test, n_classes, n_cand, 1, flags, xw1, sr, gs, &p1);
  plan_search(s.F, n_train, n_test, n_classes, n_cand, 1, flags, xw1, sr, gs, &p1n, false);
  if (p1n.total > p1.total) p1 = p1n;
  if (min_bytes) *min_bytes = p1.total;
  int kc = n_cand;
  if (budget_bytes) {
    const size_t room = budget_bytes > LB_WS_HEAD ? budget_bytes - LB_WS_HEAD : 0;
    kc = fit_chunk(s.F, n_train, n_test, n_classes, n_cand, flags, xw1, sr, gs, room);
    const int kn = fit_chunk(s.F, n_train, n_test, n_classes, n_cand, flags, xw1, sr, gs, room, false);
    if (kn < kc) kc = kn;                                  // a size both settings of LBCNN_OPT_DUAL_TRICK can run in
    if (kc < 1) kc = 1;
  }
  SearchPlan p, pn;
  plan_search(s.F, n_train, n_test, n_classes, n_cand, kc, flags, xw1, sr, gs, &p);
  plan_search(s.F, n_train, n_test, n_classes, n_cand, kc, flags, xw1, sr, gs, &pn, false);   // LBCNN_OPT_DUAL_TRICK off: the larger one fits both
  if (pn.total > p.total) p = pn;
  if (min_bytes) *min_bytes += LB_WS_HEAD;
  *bytes = p.total + LB_WS_HEAD;
  return LBCNN_OK;
}

int lbcnn_expand_workspace_bytes(lbcnn_handle_t h, const lbcnn_arch_t* arch, int32_t n_cand, int32_t has_bias, size_t* bytes) {
  if (!h || !bytes || n_cand < 1) return LBCNN_ERR_INVALID_ARG;
  ArchShape s;
  const int rc = lb_arch_shape(arch, &s);
  if (rc) return rc;
  *bytes = lb_expand_ws_bytes(h, s, has_bias != 0, n_cand);
  if (*bytes) *bytes += LB_WS_HEAD;
  return LBCNN_OK;
}

int lbcnn_expand(lbcnn_handle_t h, const lbcnn_arch_t* arch, const uint8_t* d_images, int64_t n, const int8_t* d_kernels,
                 const int32_t* d_bias, int32_t n_cand, float* d_H, void* stream) {
  if (!h || !arch || !d_images || !d_kernels || !d_H || n < 1 || n_cand < 1) return LBCNN_ERR_INVALID_ARG;
  ArchShape s;
  const int rc = lb_arch_shape(arch, &s);
  if (rc) return rc;
  return lb_launch_expand(h, s, arch->feature_scale, d_images, n, d_kernels, d_bias, n_cand, d_H, lb_ws_base(h), lb_ws_avail(h),
                          (cudaStream_t)stream);
}

int lbcnn_fit_workspace_bytes(int64_t n, int64_t F, int32_t n_classes, int32_t n_cand, uint32_t flags, size_t* bytes) {
  if (!bytes || n < 1 || F < 1 || n_classes < 2 || n_cand < 1) return LBCNN_ERR_INVALID_ARG;
  FitPlan p;
  lb_fit_plan(n, F, n_classes, n_cand, flags, &p);
  *bytes = p.total + LB_WS_HEAD;
  return LBCNN_OK;
}

int lbcnn_expand_path(lbcnn_handle_t h, const lbcnn_arch_t* arch, int32_t has_bias, int32_t* path) {
  if (!h || !arch || !path) return LBCNN_ERR_INVALID_ARG;
  ArchShape s;
  const int rc = lb_arch_shape(arch, &s);
  if (rc) return rc;
  *path = (!h->force_simt_expand && lb_expand_tc_usable(h, s, has_bias != 0)) ? LBCNN_EXPAND_TENSOR : LBCNN_EXPAND_SIMT;
  return LBCNN_OK;
}

int lbcnn_elm_fit(lbcnn_handle_t h, const float* d_H, int64_t n, int64_t F, float h_scale, uint32_t flags,
                  const int32_t* d_labels, int32_t n_classes, float C, int32_t n_cand, float* d_W, int32_t* d_info,
                  void* stream) {
  if (!h || !d_H || !d_labels || !d_W || !d_info || n < 1 || F < 1 || n_classes < 2 || n_cand < 1) return LBCNN_ERR_INVALID_ARG;
  if (!(C > 0.0f) || !(h_scale > 0.0f)) return LBCNN_ERR_INVALID_ARG;
  if (n > 2147483647LL || F > 2147483647LL || n_cand > 65535) return LBCNN_ERR_INVALID_ARG;
  FitPlan p;
  lb_fit_plan(n, F, n_classes, n_cand, flags, &p);
  if (!h->ws || lb_ws_avail(h) < p.total) return LBCNN_ERR_WORKSPACE;
  return lb_launch_fit(h, lb_ws_base(h), p, d_H, n, F, h_scale, d_labels, n_classes, C, n_cand, d_W, d_info, (cudaStream_t)stream);
}

int lbcnn_elm_score(lbcnn_handle_t h, const float* d_H, int64_t n, int64_t F, float h_scale, const float* d_W,
                    int32_t n_classes, const int32_t* d_labels, int32_t n_cand, int32_t* d_pred, int32_t* d_correct,
                    void* stream) {
  if (!h || !d_H || !d_W || n < 1 || F < 1 || n_classes < 2 || n_cand < 1) return LBCNN_ERR_INVALID_ARG;
  if (d_correct && !d_labels) return LBCNN_ERR_INVALID_ARG;
  if (n > 2147483647LL || F > 2147483647LL || n_cand > 65535) return LBCNN_ERR_INVALID_ARG;
  if (h->scorer == LBCNN_SCORER_TENSOR && lb_score_tc_usable(d_H, n, F, n_classes, n_cand)) {
    if (!h->ws || lb_ws_avail(h) < lb_score_tc_ws_bytes(n, F, n_classes, n_cand)) return LBCNN_ERR_WORKSPACE;
    return lb_launch_score_tc(h, lb_ws_base(h), d_H, n, F, h_scale, d_W, n_classes, d_labels, n_cand, d_pred, d_correct,
                              (cudaStream_t)stream);
  }
  return lb_launch_score(h, d_H, n, F, h_scale, d_W, n_classes, d_labels, n_cand, d_pred, d_correct, (cudaStream_t)stream);
}

int lbcnn_quantize_output_layer(lbcnn_handle_t h, const float* d_W, int64_t F, int32_t n_classes, int32_t n_cand, int32_t bits,
                                int8_t* d_Wq, float* d_scale, void* stream) {
  if (!h || !d_W || !d_Wq || !d_scale || F < 1 || n_classes < 2 || n_cand < 1 || n_cand > 65535) return LBCNN_ERR_INVALID_ARG;
  if (bits < 2 || bits > 8) return LBCNN_ERR_INVALID_ARG;
  return lb_launch_quantize_w(h, d_W, F, n_classes, n_cand, bits, d_Wq, d_scale, (cudaStream_t)stream);
}

int lbcnn_elm_score_q(lbcnn_handle_t h, const float* d_H, int64_t n, int64_t F, const int8_t* d_Wq, int32_t n_classes,
                      const int32_t* d_labels, int32_t n_cand, int32_t* d_pred, int32_t* d_correct, void* stream) {
  if (!h || !d_H || !d_Wq || n < 1 || F < 1 || n_classes < 2 || n_cand < 1) return LBCNN_ERR_INVALID_ARG;
  if (d_correct && !d_labels) return LBCNN_ERR_INVALID_ARG;
  if (!lb_score_tc_usable(d_H, n, F, n_classes, n_cand)) return LBCNN_ERR_SHAPE;
  if (!h->ws || lb_ws_avail(h) < lb_score_tc_ws_bytes(n, F, n_classes, n_cand)) return LBCNN_ERR_WORKSPACE;
  return lb_launch_score_q8(h, lb_ws_base(h), d_H, n, F, d_Wq, n_classes, d_labels, n_cand, d_pred, d_correct, (cudaStream_t)stream);
}

int lbcnn_evolve_candidates(lbcnn_handle_t h, const int8_t* d_kernels, const float* d_acc, int32_t n_cand, int64_t n_weights,
                            int32_t n_elite, uint32_t mut_ppm, uint64_t seed, uint32_t generation, int8_t* d_next, void* stream) {
  if (!h || !d_kernels || !d_acc || !d_next || n_cand < 1 || n_cand > 16384 || n_weights < 1) return LBCNN_ERR_INVALID_ARG;
  if (n_elite < 0 || n_elite > n_cand || mut_ppm > 1000000u || d_next == d_kernels) return LBCNN_ERR_INVALID_ARG;
  if (!h->ws || lb_ws_avail(h) < (size_t)n_cand * 8) return LBCNN_ERR_WORKSPACE;
  return lb_launch_evolve(h, lb_ws_base(h), d_kernels, d_acc, n_cand, n_weights, n_elite, mut_ppm, seed, generation, d_next,
                          (cudaStream_t)stream);
}

int lbcnn_refine_workspace_bytes(int64_t F, int32_t n_classes, const lbcnn_refine_t* cfg, size_t* bytes) {
  if (!bytes || !cfg || F < 1 || n_classes < 2 || cfg->epochs < 0 || cfg->batch < 1) return LBCNN_ERR_INVALID_ARG;
  *bytes = lb_refine_ws_bytes(F, n_classes, cfg->batch, cfg->epochs) + LB_WS_HEAD;
  return LBCNN_OK;
}

int lbcnn_refine_output_layer(lbcnn_handle_t h, const float* d_H, int64_t n, int64_t F, float h_scale, const int32_t* d_labels,
                              int32_t n_classes, const lbcnn_refine_t* cfg, float* d_W, float* d_loss, void* stream) {
  if (!h || !d_H || !d_labels || !cfg || !d_W || n < 1 || F < 1 || n_classes < 2) return LBCNN_ERR_INVALID_ARG;
  if (cfg->epochs < 0 || cfg->batch < 1 || !(cfg->lr > 0.0f) || !(h_scale > 0.0f) || n > 2147483647LL || F > 2147483647LL)
    return LBCNN_ERR_INVALID_ARG;
  if (!(cfg->beta1 >= 0.0f && cfg->beta1 < 1.0f && cfg->beta2 >= 0.0f && cfg->beta2 < 1.0f && cfg->eps >= 0.0f)) return LBCNN_ERR_INVALID_ARG;
  if (!h->ws || lb_ws_avail(h) < lb_refine_ws_bytes(F, n_classes, cfg->batch, cfg->epochs)) return LBCNN_ERR_WORKSPACE;
  return lb_launch_refine(h, lb_ws_base(h), d_H, n, F, h_scale, d_labels, n_classes, *cfg, d_W, d_loss, (cudaStream_t)stream);
}

int lbcnn_score_workspace_bytes(int64_t n, int64_t F, int32_t n_classes, int32_t n_cand, size_t* bytes) {
  if (!bytes || n < 1 || F < 1 || n_classes < 2 || n_cand < 1) return LBCNN_ERR_INVALID_ARG;
  *bytes = lb_score_tc_ws_bytes(n, F, n_classes, n_cand) + LB_WS_HEAD;
  return LBCNN_OK;
}

}  // extern "C"

// the search loop on device buffers, scratch taken from [ws, ws + ws_bytes)
static int search_impl(lbcnn_handle_t h, void* ws, size_t ws_bytes, const lbcnn_arch_t* arch, const uint8_t* d_train,
                       const int32_t* d_train_labels, int64_t n_train, const uint8_t* d_test,
                       const int32_t* d_test_labels, int64_t n_test, int32_t n_classes, float C,
                       const int8_t* d_kernels, const int32_t* d_bias, int32_t n_cand, float* d_acc,
                       int32_t* d_correct, int32_t* d_info, int32_t* d_best, float* d_W_best, void* stream) {
  if (!h || !arch || !d_train || !d_train_labels || !d_test || !d_test_labels || !d_kernels || !d_acc || !d_correct ||
      !d_info || !d_best)
    return LBCNN_ERR_INVALID_ARG;
  if (n_train < 1 || n_test < 1 || n_classes < 2 || n_cand < 1 || !(C > 0.0f) || !(arch->feature_scale > 0.0f))
    return LBCNN_ERR_INVALID_ARG;
  ArchShape s;
  int rc = lb_arch_shape(arch, &s);
  if (rc) return rc;
  if (n_cand > 65535 * 64) return LBCNN_ERR_INVALID_ARG;
  if (!ws) return LBCNN_ERR_WORKSPACE;
  const uint32_t fflags = search_fit_flags(s, d_bias != nullptr);
  const size_t xw1 = lb_expand_ws_bytes(h, s, d_bias != nullptr, 1);
  const int64_t sr = h->stream_rows;
  const bool want_kt = h->dual_trick != 0 && h->scorer != LBCNN_SCORER_FP64;
  const size_t gs = gather_slot_bytes(s);
  int kc = fit_chunk(s.F, n_train, n_test, n_classes, n_cand, fflags, xw1, sr, gs, ws_bytes, want_kt);
  if (kc < 1) return LBCNN_ERR_WORKSPACE;
  if (kc > 65535) kc = 65535;                          // grid.y / grid.z of the batched kernels
  SearchPlan p;
  plan_search(s.F, n_train, n_test, n_classes, n_cand, kc, fflags, xw1, sr, gs, &p, want_kt);
  char* base = reinterpret_cast<char*>(ws);
  float* Htr = reinterpret_cast<float*>(base + p.htr_off);
  float* Hte = reinterpret_cast<float*>(base + p.hte_off);
  float* Wall = reinterpret_cast<float*>(base + p.w_off);
  cudaStream_t st = (cudaStream_t)stream;
  const float hs = arch->feature_scale;
  const int64_t wel = s.F * n_classes;
  const int64_t px = (int64_t)s.L[0].hin * s.L[0].win * s.L[0].cin;      // bytes of one image
  for (int k0 = 0; k0 < n_cand; k0 += kc) {
    const int kn = (n_cand - k0 < kc) ? n_cand - k0 : kc;
    const int8_t* ker = d_kernels + (int64_t)k0 * s.n_weights;
    const int32_t* bias = d_bias ? d_bias + (int64_t)k0 * s.n_bias : nullptr;
    float* Wk = Wall + (int64_t)k0 * wel;
    const bool tc_score = (fflags & LBCNN_H_INTEGER) && h->scorer != LBCNN_SCORER_FP64 &&
                          lb_score_tc_usable(Hte, p.nte_ws, s.F, n_classes, kn) &&
                          (h->scorer == LBCNN_SCORER_TENSOR || lb_score_tc_worthwhile(n_test, s.F, n_classes, kn));
    FitPlan fp;
    if (p.dual_kt) {
      // dual branch through the kernel trick: one buffer [candidate][train rows | test rows][F]; the exact Gram of the stack
      // holds the cross-Gram H_te U^T, the factorisation turns it into the logits (fit.cu); W only for the best, afterwards
      const int64_t n_all = n_train + n_test;
      lb_fit_plan(n_train, s.F, n_classes, kn, fflags, &fp, 0, n_test);
      fp.allow_tc = arch_allows_tc_solver(s) ? 1 : 0;
      rc = lb_launch_expand(h, s, 1.0f, d_train, n_train, ker, bias, kn, Htr, base + p.xw_off, xw1 * (size_t)kn, st, false, n_all);
      if (rc) return rc;
      rc = lb_launch_expand(h, s, 1.0f, d_test, n_test, ker, bias, kn, Htr + n_train * s.F, base + p.xw_off, xw1 * (size_t)kn, st, true, n_all);
      if (rc) return rc;
      const DualScore dsc{d_test_labels, d_correct + k0};
      rc = lb_launch_fit(h, base + p.fit_off, fp, Htr, n_train, s.F, hs, d_train_labels, n_classes, C, kn, Wk, d_info + k0, st, nullptr, &dsc);
      if (rc) return rc;
      if (k0 + kn < n_cand) continue;                  // more chunks to come
      rc = lb_launch_finish(h, d_correct, d_info, n_test, n_cand, d_acc, d_best, nullptr, wel, nullptr, st);
      if (rc) return rc;
      if (!d_W_best) return LBCNN_OK;
      if (kc >= n_cand)                                // one chunk: the best candidate's features and solution are still here
        return lb_launch_w_best_dual(h, base + p.fit_off, fp, d_best, Htr, n_train, s.F, hs, n_classes, d_W_best, st);
      // several chunks: the best candidate's chunk may be gone and its index exists on the device only.  Its kernel set is
      // gathered into a slot of its own and the candidate is fitted once more, alone, with the explicit W = H^T Z.
      int8_t* gker = reinterpret_cast<int8_t*>(base + p.gs_off);
      int32_t* gbias = reinterpret_cast<int32_t*>(base + p.gs_off + lb_align_up(s.n_weights, 256));
      int32_t* ginfo = reinterpret_cast<int32_t*>(base + p.gs_off + lb_align_up((int64_t)gs, 256));
      rc = lb_launch_gather_best(h, d_best, d_kernels, s.n_weights, d_bias, s.n_bias, gker, gbias, st);
      if (rc) return rc;
      FitPlan f1;
      lb_fit_plan(n_train, s.F, n_classes, 1, fflags, &f1);
      f1.allow_tc = fp.allow_tc;
      if (f1.total > p.fit.total) return LBCNN_ERR_WORKSPACE;
      rc = lb_launch_expand(h, s, 1.0f, d_train, n_train, gker, d_bias ? gbias : nullptr, 1, Htr, base + p.xw_off, xw1, st, false);
      if (rc) return rc;
      return lb_launch_fit(h, base + p.fit_off, f1, Htr, n_train, s.F, hs, d_train_labels, n_classes, C, 1, d_W_best, ginfo, st);
    }
    lb_fit_plan(n_train, s.F, n_classes, kn, fflags, &fp, p.ntr_ws);
    fp.allow_tc = arch_allows_tc_solver(s) ? 1 : 0;
    // E1-E4 with scale 1: H holds the exact integers; the scale enters the fit and the score as h_scale.
    // Streamed ("limited GPU-RAM"): the train set passes through in chunks of
    // ntr_ws samples whose exact integer Grams (and fused right-hand sides) add up in A -- H of the whole set never exists.
    for (int64_t r0 = 0; r0 < n_train; r0 += p.ntr_ws) {
      const int64_t nr = (n_train - r0 < p.ntr_ws) ? n_train - r0 : p.ntr_ws;
      rc = lb_launch_expand(h, s, 1.0f, d_train + r0 * px, nr, ker, bias, kn, Htr, base + p.xw_off, xw1 * (size_t)kn, st, r0 > 0);
      if (rc) return rc;
      if (p.stream) {
        const FitStream fs{1, r0 == 0 ? 1 : 0, r0 + nr >= n_train ? 1 : 0};
        rc = lb_launch_fit(h, base + p.fit_off, fp, Htr, nr, s.F, hs, d_train_labels + r0, n_classes, C, kn, Wk, d_info + k0, st, &fs);
        if (rc) return rc;
      }
    }
    {
      const FitStream fs{2, 0, 0};
      rc = lb_launch_fit(h, base + p.fit_off, fp, Htr, n_train, s.F, hs, d_train_labels, n_classes, C, kn, Wk, d_info + k0, st,
                         p.stream ? &fs : nullptr);
      if (rc) return rc;
    }
    for (int64_t r0 = 0; r0 < n_test; r0 += p.nte_ws) {
      const int64_t nr = (n_test - r0 < p.nte_ws) ? n_test - r0 : p.nte_ws;
      rc = lb_launch_expand(h, s, 1.0f, d_test + r0 * px, nr, ker, bias, kn, Hte, base + p.xw_off, xw1 * (size_t)kn, st, true);
      if (rc) return rc;
      if (tc_score)
        rc = lb_launch_score_tc(h, base + p.sc_off, Hte, nr, s.F, hs, Wk, n_classes, d_test_labels + r0, kn, nullptr, d_correct + k0, st,
                                r0 > 0);
      else
        rc = lb_launch_score(h, Hte, nr, s.F, hs, Wk, n_classes, d_test_labels + r0, kn, nullptr, d_correct + k0, st, r0 > 0);
      if (rc) return rc;
    }
  }
  return lb_launch_finish(h, d_correct, d_info, n_test, n_cand, d_acc, d_best, Wall, wel, d_W_best, st);
}

// ---- host-buffer staging layout (lbcnn_search_candidates_host) ----------------------------------
namespace {
struct HostStage {
  size_t train, train_y, test, test_y, ker, bias, acc, correct, info, best, wbest, total;
};
void plan_host_stage(const ArchShape& s, int64_t n_train, int64_t n_test, int c, int n_cand, int has_bias, HostStage* p) {
  const int64_t px = (int64_t)s.L[0].hin * s.L[0].win * s.L[0].cin;
  size_t off = 0;
  auto take = [&](int64_t bytes) { size_t o = off; off += (size_t)lb_align_up(bytes, 256); return o; };
  p->train = take(n_train * px);
  p->train_y = take(n_train * 4);
  p->test = take(n_test * px);
  p->test_y = take(n_test * 4);
  p->ker = take((int64_t)n_cand * s.n_weights);
  p->bias = take(has_bias ? (int64_t)n_cand * s.n_bias * 4 : 0);
  p->acc = take((int64_t)n_cand * 4);
  p->correct = take((int64_t)n_cand * 4);
  p->info = take((int64_t)n_cand * 4);
  p->best = take(8);
  p->wbest = take(s.F * c * 4);
  p->total = off;
}
}  // namespace

extern "C" {

int lbcnn_search_candidates(lbcnn_handle_t h, const lbcnn_arch_t* arch, const uint8_t* d_train,
                            const int32_t* d_train_labels, int64_t n_train, const uint8_t* d_test,
                            const int32_t* d_test_labels, int64_t n_test, int32_t n_classes, float C,
                            const int8_t* d_kernels, const int32_t* d_bias, int32_t n_cand, float* d_acc,
                            int32_t* d_correct, int32_t* d_info, int32_t* d_best, float* d_W_best, void* stream) {
  if (!h) return LBCNN_ERR_INVALID_ARG;
  return search_impl(h, lb_ws_base(h), lb_ws_avail(h), arch, d_train, d_train_labels, n_train, d_test, d_test_labels, n_test,
                     n_classes, C, d_kernels, d_bias, n_cand, d_acc, d_correct, d_info, d_best, d_W_best, stream);
}

int lbcnn_host_staging_bytes(const lbcnn_arch_t* arch, int64_t n_train, int64_t n_test, int32_t n_classes,
                             int32_t n_cand, int32_t has_bias, size_t* bytes) {
  if (!bytes || n_train < 1 || n_test < 1 || n_classes < 2 || n_cand < 1) return LBCNN_ERR_INVALID_ARG;
  ArchShape s;
  const int rc = lb_arch_shape(arch, &s);
  if (rc) return rc;
  HostStage p;
  plan_host_stage(s, n_train, n_test, n_classes, n_cand, has_bias, &p);
  *bytes = p.total;
  return LBCNN_OK;
}

int lbcnn_search_candidates_host(lbcnn_handle_t h, const lbcnn_arch_t* arch, const uint8_t* h_train,
                                 const int32_t* h_train_labels, int64_t n_train, const uint8_t* h_test,
                                 const int32_t* h_test_labels, int64_t n_test, int32_t n_classes, float C,
                                 const int8_t* h_kernels, const int32_t* h_bias, int32_t n_cand, float* h_acc,
                                 int32_t* h_correct, int32_t* h_info, int32_t* h_best, float* h_W_best, void* stream) {
  if (!h || !arch || !h_train || !h_train_labels || !h_test || !h_test_labels || !h_kernels || !h_acc || !h_correct ||
      !h_info || !h_best)
    return LBCNN_ERR_INVALID_ARG;
  if (n_train < 1 || n_test < 1 || n_classes < 2 || n_cand < 1) return LBCNN_ERR_INVALID_ARG;
  ArchShape s;
  int rc = lb_arch_shape(arch, &s);
  if (rc) return rc;
  HostStage p;
  plan_host_stage(s, n_train, n_test, n_classes, n_cand, h_bias != nullptr, &p);
  if (!h->ws || lb_ws_avail(h) <= p.total) return LBCNN_ERR_WORKSPACE;
  char* base = lb_ws_base(h);
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t px = (int64_t)s.L[0].hin * s.L[0].win * s.L[0].cin;
  LB_CUDA_OK(cudaMemcpyAsync(base + p.train, h_train, (size_t)(n_train * px), cudaMemcpyHostToDevice, st));
  LB_CUDA_OK(cudaMemcpyAsync(base + p.train_y, h_train_labels, (size_t)n_train * 4, cudaMemcpyHostToDevice, st));
  LB_CUDA_OK(cudaMemcpyAsync(base + p.test, h_test, (size_t)(n_test * px), cudaMemcpyHostToDevice, st));
  LB_CUDA_OK(cudaMemcpyAsync(base + p.test_y, h_test_labels, (size_t)n_test * 4, cudaMemcpyHostToDevice, st));
  LB_CUDA_OK(cudaMemcpyAsync(base + p.ker, h_kernels, (size_t)n_cand * s.n_weights, cudaMemcpyHostToDevice, st));
  if (h_bias)
    LB_CUDA_OK(cudaMemcpyAsync(base + p.bias, h_bias, (size_t)n_cand * s.n_bias * 4, cudaMemcpyHostToDevice, st));
  float* d_acc = reinterpret_cast<float*>(base + p.acc);
  int32_t* d_correct = reinterpret_cast<int32_t*>(base + p.correct);
  int32_t* d_info = reinterpret_cast<int32_t*>(base + p.info);
  int32_t* d_best = reinterpret_cast<int32_t*>(base + p.best);
  float* d_wb = h_W_best ? reinterpret_cast<float*>(base + p.wbest) : nullptr;
  rc = search_impl(h, base + p.total, lb_ws_avail(h) - p.total, arch, reinterpret_cast<const uint8_t*>(base + p.train),
                   reinterpret_cast<const int32_t*>(base + p.train_y), n_train,
                   reinterpret_cast<const uint8_t*>(base + p.test), reinterpret_cast<const int32_t*>(base + p.test_y),
                   n_test, n_classes, C, reinterpret_cast<const int8_t*>(base + p.ker),
                   h_bias ? reinterpret_cast<const int32_t*>(base + p.bias) : nullptr, n_cand, d_acc, d_correct, d_info,
                   d_best, d_wb, stream);
  if (rc) return rc;
  LB_CUDA_OK(cudaMemcpyAsync(h_acc, d_acc, (size_t)n_cand * 4, cudaMemcpyDeviceToHost, st));
  LB_CUDA_OK(cudaMemcpyAsync(h_correct, d_correct, (size_t)n_cand * 4, cudaMemcpyDeviceToHost, st));
  LB_CUDA_OK(cudaMemcpyAsync(h_info, d_info, (size_t)n_cand * 4, cudaMemcpyDeviceToHost, st));
  LB_CUDA_OK(cudaMemcpyAsync(h_best, d_best, 8, cudaMemcpyDeviceToHost, st));
  if (h_W_best) LB_CUDA_OK(cudaMemcpyAsync(h_W_best, d_wb, (size_t)(s.F * n_classes) * 4, cudaMemcpyDeviceToHost, st));
  LB_CUDA_OK(cudaStreamSynchronize(st));
  return LBCNN_OK;
}

}  // extern "C"
