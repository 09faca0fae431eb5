// internal.h -- declarations shared by the translation units of liblbcnn (CUDA path only;
// nothing here is used by, or shared with, oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/lbcnn.h"
#include <vector>

struct LbPhaseRec { int phase; cudaEvent_t start, stop; };

struct lbcnn_handle_s {
  int device;
  int n_sm;
  int max_smem_optin;  // bytes of dynamic shared memory one CTA may opt in to
  void* ws;
  size_t ws_bytes;
  int64_t launches;
  int force_simt_expand;            // testing (lbcnn_set_option): keep the expander on the SIMT kernel
  int solver;                       // LBCNN_SOLVER_* (lbcnn_set_option)
  int panel;                        // panel width of the blocked Cholesky when its trailing updates run on tcgen05
  int deflate;                      // ... with the first block column's update kept in fp64 (common-mode deflation)
  int scorer;                       // LBCNN_SCORER_* (lbcnn_set_option)
  int mid_panel;                    // width of the fp64-stepped blocks inside a panel (three-level factorisation); 0 = two levels
  int64_t stream_rows;              // search driver: samples expanded / accumulated per chunk (0 = all at once)
  int dual_trick;                   // search driver, dual branch: score through the cross-Gram (kernel trick), W for the best only
  int profiling;                    // record CUDA events around each phase of the path
  std::vector<LbPhaseRec> recs;
};

// RAII phase marker: records start/stop events on the stream when profiling is on
struct LbPhase {
  lbcnn_handle_s* h; cudaStream_t st; LbPhaseRec r; bool on;
  LbPhase(lbcnn_handle_s* h_, int phase, cudaStream_t st_, bool enable = true) : h(h_), st(st_), on(h_->profiling != 0 && enable) {
    if (on) { r.phase = phase; cudaEventCreate(&r.start); cudaEventCreate(&r.stop); cudaEventRecord(r.start, st); }
  }
  void stop() { if (on) { cudaEventRecord(r.stop, st); h->recs.push_back(r); on = false; } }
  ~LbPhase() { stop(); }
};

#define LB_CUDA_OK(expr)                                  \
  do {                                                    \
    cudaError_t e__ = (expr);                             \
    if (e__ != cudaSuccess) return LBCNN_ERR_CUDA;        \
  } while (0)

// The first LB_WS_HEAD bytes of the caller's workspace hold the library's measurement counters (zeroed by
// lbcnn_set_workspace): [0] int8 multiply-adds issued by the Gram kernel, [1] by the Cholesky trailing updates.
constexpr size_t LB_WS_HEAD = 256;
static inline char* lb_ws_base(const lbcnn_handle_s* h) { return h->ws ? reinterpret_cast<char*>(h->ws) + LB_WS_HEAD : nullptr; }
static inline size_t lb_ws_avail(const lbcnn_handle_s* h) { return h->ws_bytes > LB_WS_HEAD ? h->ws_bytes - LB_WS_HEAD : 0; }
static inline unsigned long long* lb_ws_counter(const lbcnn_handle_s* h, int i) {
  return h->ws ? reinterpret_cast<unsigned long long*>(h->ws) + i : nullptr;
}

// largest |u| three balanced radix-256 int8 digits represent: 127 + 127*256 + 127*65536
constexpr int64_t LB_H_INTEGER_MAX = 8355711;

static inline int64_t lb_align_up(int64_t x, int64_t a) { return (x + a - 1) / a * a; }

// ---- host shape logic (api.cu) -------------------------------------------------------------
struct LayerShape {
  int conv_type, nk, k, act, pk, ps, pp, cover;
  int cin, cout, hin, win, hout, wout;
  int64_t w_off, b_off;   // offsets of this layer inside one candidate's kernel set / bias set
};
struct ArchShape {
  int n_layers;
  LayerShape L[3];
  int64_t F, n_weights, n_bias;
  int64_t max_abs;        // bound on |integer feature| (255 * prod k^2 Cin), saturated at 2^62
};
int lb_pool_out(int n, int k, int s, int p, int cover_all);
int lb_arch_shape(const lbcnn_arch_t* a, ArchShape* s);

// ---- expander (expand.cu) ------------------------------------------------------------------
// xw / xw_bytes: caller scratch of lb_expand_ws_bytes() bytes (the tensor-core kernel's prepared operands)
size_t lb_expand_ws_bytes(const lbcnn_handle_s* h, const ArchShape& s, bool has_bias, int n_cand);
// prepared: xw already holds these candidates' operands from an earlier call (the driver expands the train and the test
// set with the same kernel sets): the re-layout kernel is not launched again
int lb_launch_expand(lbcnn_handle_s* h, const ArchShape& s, float feature_scale, const uint8_t* d_images, int64_t n,
                     const int8_t* d_kernels, const int32_t* d_bias, int n_cand, float* d_H, void* xw, size_t xw_bytes,
                     cudaStream_t st, bool prepared = false, int64_t out_rows = 0);   // out_rows: rows per candidate of d_H (0 = n)

// tensor-core expander (expand_tc.cu): FULL convolutions, non-overlapping pooling, 1-2 layers, no bias
bool lb_expand_tc_usable(const lbcnn_handle_s* h, const ArchShape& s, bool has_bias);
size_t lb_expand_tc_ws_bytes(const lbcnn_handle_s* h, const ArchShape& s, bool has_bias, int n_cand);
int lb_launch_expand_tc(lbcnn_handle_s* h, const ArchShape& s, float feature_scale, const uint8_t* d_images, int64_t n,
                        const int8_t* d_kernels, int n_cand, float* d_H, void* xw, size_t xw_bytes, cudaStream_t st,
                        bool prepared = false, int64_t out_rows = 0);

// ---- fit (fit.cu) --------------------------------------------------------------------------
struct FitPlan {
  int primal;            // 1: F x F system, 0: n x n system
  int64_t dim;           // system dimension
  int64_t rows;          // dim + n_classes (right-hand sides appended as rows)
  size_t a_bytes;        // per candidate: rows * dim doubles
  size_t perm_off, off_off, a_off, tc_off, linv_off, stc_off, total; // offsets inside the fit workspace
  int64_t n_extra;       // dual branch, search driver: test samples stacked behind the train samples (cross-Gram rows in A)
  size_t lg_off;         // ... and their logits [n_cand][n_extra][n_classes] fp64
  int allow_tc;          // LBCNN_SOLVER_AUTO may take the tensor-core updates (set by the search driver when the architecture
                         // cannot produce (anti)collinear features; lbcnn_elm_fit leaves it 0: unknown data -> all-fp64)
  int stc_kmax;          // widest panel the tensor-core trailing update is planned for (0: no scratch reserved)
  int use_tc;            // Gram on the tensor pipe (exact int8-digit path, gram_tc.cu)
  int fuse_rhs;          // ... which then also produces the right-hand side (one-hot label columns)
};
// n_ws: rows of H resident at once (streamed Gram: the digit planes are sized for one chunk of samples); 0 = n
void lb_fit_plan(int64_t n, int64_t F, int n_classes, int n_cand, uint32_t flags, FitPlan* p, int64_t n_ws = 0, int64_t n_extra = 0);
// streamed fit: stage 1 = add one chunk of samples to the Gram (+ fused right-hand side), stage 2 = solve
struct FitStream { int stage; int first_chunk; int last_chunk; };
// dual branch scored through the kernel trick (plan.n_extra test rows stacked behind the train rows of d_H): logits =
// (H_te U^T) Z come out of the factorisation's appended rows; W is not formed for every candidate
struct DualScore { const int32_t* te_labels; int32_t* correct; };
int lb_launch_w_best_dual(lbcnn_handle_s* h, void* ws, const FitPlan& p, const int32_t* d_best, const float* d_Hall, int64_t n,
                          int64_t F, float h_scale, int n_classes, float* d_W_best, cudaStream_t st);
int lb_launch_fit(lbcnn_handle_s* h, void* ws, const FitPlan& p, const float* d_H, int64_t n, int64_t F, float h_scale,
                  const int32_t* d_labels, int n_classes, float C, int n_cand, float* d_W, int32_t* d_info,
                  cudaStream_t st, const FitStream* fs = nullptr, const DualScore* ds = nullptr);

// ---- exact integer Gram on tcgen05 (gram_tc.cu) ---------------------------------------------------
constexpr int64_t LB_GRAM_TC_MAX_K = 43690;   // longest contraction whose int32 accumulators stay exact: 3 * 128^2 * k < 2^31
bool lb_gram_tc_usable(int64_t n, int64_t F, bool primal);
size_t lb_gram_tc_ws_bytes(int64_t n, int64_t F, int n_cand, int c_aug);
bool lb_gram_tc_fuse_rhs(int64_t F, int n_classes);   // right-hand side as one-hot columns of the Gram's digit plane 0
int lb_launch_gram_tc(lbcnn_handle_s* h, void* ws, const float* d_U, int64_t n, int64_t F, int n_cand, double lam, double* A,
                      long long a_stride, long long ld, bool primal, const int32_t* d_labels, int n_classes, int32_t* d_info,
                      cudaStream_t st, bool accumulate = false, bool add_lam = true,    // streamed: A += this chunk's Gram; ridge with the last chunk
                      int64_t n_rows = 0, int rshift = 0);   // dual: n_rows >= n samples in H (test rows behind the train rows)

constexpr int LB_STC_KMAX = 1024;      // widest panel (digit-plane pitch)
constexpr int LB_STC_MIN_DIM = 512;    // systems below this never reserve the scratch
constexpr int LB_STC_AUTO_DIM = 1024;  // LBCNN_SOLVER_AUTO takes the tensor-core updates from this dimension on
// ---- Cholesky trailing updates on tcgen05 (chol_tc.cu) ------------------------------------------------
struct CholTcCtx {
  alignas(64) unsigned char tmap[128];   // CUtensorMap of the digit planes
  int8_t* planes; double* rscale; int pitch;
  int64_t rows, dim; int n_cand;
  double* A; long long a_stride, ld;
  unsigned long long* ops;
};
size_t lb_chol_tc_ws_bytes(int64_t rows, int n_cand, int kmax);
int lb_chol_tc_begin(lbcnn_handle_s* h, void* ws, int64_t rows, int64_t dim, int n_cand, int kmax, double* A,
                     long long a_stride, long long ld, unsigned long long* ops, CholTcCtx* ctx);
int lb_chol_tc_update(lbcnn_handle_s* h, const CholTcCtx& ctx, int r0, int c1, int k0, int K, cudaStream_t st);

// ---- score (score.cu) ----------------------------------------------------------------------
// keep_correct: add to d_correct instead of starting from zero (streamed scoring of test-set chunks)
int lb_launch_score(lbcnn_handle_s* h, const float* d_H, int64_t n, int64_t F, float h_scale, const float* d_W,
                    int n_classes, const int32_t* d_labels, int n_cand, int32_t* d_pred, int32_t* d_correct,
                    cudaStream_t st, bool keep_correct = false);
// tensor-core scorer (score_tc.cu): integer-valued features, up to 128 classes; scratch from the caller's workspace
bool lb_score_tc_usable(const float* d_H, int64_t n, int64_t F, int n_classes, int n_cand);
bool lb_score_tc_worthwhile(int64_t n, int64_t F, int n_classes, int n_cand);
size_t lb_score_tc_ws_bytes(int64_t n, int64_t F, int n_classes, int n_cand);
int lb_launch_score_tc(lbcnn_handle_s* h, void* ws, const float* d_H, int64_t n, int64_t F, float h_scale, const float* d_W,
                       int n_classes, const int32_t* d_labels, int n_cand, int32_t* d_pred, int32_t* d_correct,
                       cudaStream_t st, bool keep_correct = false);
// <= 8-bit output layer (score_tc.cu): per-candidate symmetric quantisation of W, and S1 with exact integer logits
int lb_launch_quantize_w(lbcnn_handle_s* h, const float* d_W, int64_t F, int n_classes, int n_cand, int bits, int8_t* d_Wq,
                         float* d_scale, cudaStream_t st);
int lb_launch_score_q8(lbcnn_handle_s* h, void* ws, const float* d_H, int64_t n, int64_t F, const int8_t* d_Wq, int n_classes,
                       const int32_t* d_labels, int n_cand, int32_t* d_pred, int32_t* d_correct, cudaStream_t st);
// one generation of the genetic candidate generator (evolve.cu); ws: 8 * n_cand bytes of scratch
int lb_launch_evolve(lbcnn_handle_s* h, void* ws, const int8_t* d_kernels, const float* d_acc, int n_cand, int64_t n_weights,
                     int n_elite, uint32_t mut_ppm, uint64_t seed, uint32_t generation, int8_t* d_next, cudaStream_t st);
// gradient refinement of the output layer (refine.cu)
size_t lb_refine_ws_bytes(int64_t F, int n_classes, int batch, int epochs);
int lb_launch_refine(lbcnn_handle_s* h, void* ws, const float* d_H, int64_t n, int64_t F, float h_scale, const int32_t* d_labels,
                     int c, const lbcnn_refine_t& cfg, float* d_W, float* d_loss, cudaStream_t st);
int lb_launch_zero_i32(lbcnn_handle_s* h, int32_t* p, int64_t n, cudaStream_t st);
int lb_launch_gather_best(lbcnn_handle_s* h, const int32_t* d_best, const int8_t* d_kernels, int64_t n_weights,
                          const int32_t* d_bias, int64_t n_bias, int8_t* ker_out, int32_t* bias_out, cudaStream_t st);
int lb_launch_finish(lbcnn_handle_s* h, const int32_t* d_correct, const int32_t* d_info, int64_t n_test, int n_cand,
                     float* d_acc, int32_t* d_best, const float* d_W_all, int64_t w_elems, float* d_W_best,
                     cudaStream_t st);
