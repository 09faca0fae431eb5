/*
 * lbcnn.h -- C ABI of the B200-native LB-CNN kernel-selection inner loop (arXiv 2106.15350).
 *
 * The loop, in the paper's words (section III Cells 4-6): draw random binary
 * convolution kernels, push the (reduced) training set through 1..3 "convolution + max-pool"
 * macro-layers with those fixed kernels, flatten, fit the only
 * trainable layer -- the linear output layer "ELM0" -- by regularised least squares
 * (PAPER.md:64-74), evaluate test accuracy and keep the best kernels.
 *
 * Conventions (all entry points)
 *   - Pointers named d_* are DEVICE pointers owned by the caller (e.g. torch allocations); pointers
 *     named h_* and all struct / out-parameter pointers are HOST pointers.  The library never
 *     allocates, frees or retains device memory; ALL scratch comes from the caller-provided workspace
 *     (lbcnn_set_workspace), and a call whose scratch does not fit returns LBCNN_ERR_WORKSPACE.  (The one exception is
 *     lbcnn_evolve_candidates_static, whose scratch is a fixed array inside the library: see there.)
 *     `stream` is a cudaStream_t passed as void* (NULL = default stream).  The handle's device must be the
 *     calling thread's current device for every call that takes a stream (lbcnn_create does not change it).
 *   - Every call returns an int status (LBCNN_OK = 0 ...) and only ENQUEUES work on `stream`; it
 *     never synchronises.  Numerical failure is not a status: a non-positive Cholesky pivot j
 *     writes d_info[k] = j + 1 (LAPACK convention) for candidate k and the batch continues;
 *     d_info[k] = -1 says candidate k's features broke the LBCNN_H_INTEGER promise (see the flag).
 *   - Layouts: images uint8 NHWC "channels last"; kernel sets int8 with entries
 *     -1/+1, per candidate the layers concatenated, layer l = [n_kernels][Cin_l][k][k]; bias int32
 *     per candidate, layers concatenated, layer l = [Cout_l]; H = features, row-major
 *     [candidate][sample][F] with the C,H,W flatten order f = (o*Hout + i)*Wout + j; W = output
 *     weights row-major [candidate][F][n_classes]; labels int32 in [0, n_classes) (a label outside
 *     that range is not an error: its sample gets an all-zero target row and is never counted correct).
 *   - H here is samples x features, the transpose of the listing's H (features x samples,
 *     PAPER.md:66); the listing's H.H^T is H^T H here.
 *   - There is no CPU fallback: without a CUDA device lbcnn_create fails with LBCNN_ERR_CUDA.
 *     The shape helpers (lbcnn_feature_dim, lbcnn_kernel_set_size, lbcnn_status_string,
 *     lbcnn_version) are host-only and need no device.
 *   - Thread safety: one handle per host thread / stream.
 */
#ifndef LBCNN_H_
#define LBCNN_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
  LBCNN_OK = 0,
  LBCNN_ERR_INVALID_ARG = 1,  /* null pointer, n < 1, C <= 0, n_classes < 2, n_cand < 1 */
  LBCNN_ERR_INVALID_ARCH = 2, /* a spatial size < 1, even kernel size, pooling window with no real cell, too large for one SM's shared memory */
  LBCNN_ERR_SHAPE = 3,        /* F / channel mismatch */
  LBCNN_ERR_WORKSPACE = 4,    /* workspace absent or too small (never a hidden allocation) */
  LBCNN_ERR_CUDA = 5,         /* no device / launch or driver error */
  LBCNN_ERR_NOMEM = 6,        /* host allocation failed (lbcnn_create) */
  LBCNN_ERR_STATIC_LIMIT = 7  /* lbcnn_evolve_candidates_static only: the problem needs more scratch than the library's built-in
                                 array holds (n_cand > LBCNN_EVOLVE_STATIC_MAX_CAND); use lbcnn_evolve_candidates with a workspace */
};

enum { LBCNN_CONV_FULL = 0, LBCNN_CONV_DEPTHWISE = 1 };
enum { LBCNN_ACT_NONE = 0, LBCNN_ACT_RELU = 1 };

/* flags of lbcnn_elm_fit */
#define LBCNN_H_INTEGER 1u /* stored H values are integers with abs <= 8355711 = 127 (1 + 2^8 + 2^16), three balanced radix-256 int8 digits (the expander's output with feature_scale = 1): the Gram is then computed exactly on the tensor cores.  A candidate holding a value outside that range, or a non-integer, gets d_info[k] = -1 and no W */
#define LBCNN_FORCE_PRIMAL 2u /* testing: take the F x F branch whatever F and n are */
#define LBCNN_FORCE_DUAL 4u   /* testing: take the n x n branch */

/* One macro-layer "convolution -> (activation) -> max-pool" (listing lines 27-31).
 * Convolution: cross-correlation, stride 1, zero padding (ksize-1)/2 (pad=1 for 3x3):
 *   FULL:      z[y,x,o]     = b[o]     + sum_{c,dy,dx} w[o,c,dy,dx] * a[y+dy-p, x+dx-p, c]
 *   DEPTHWISE: z[y,x,c*M+m] = b[c*M+m] + sum_{dy,dx}   w[m,c,dy,dx] * a[y+dy-p, x+dx-p, c]
 * Pool: max over the in-image cells of window rows i*s-p .. i*s-p+k-1 (same for columns); padding never
 * wins; output size floor((n+2p-k)/s)+1, or ceil(...)+1 with cover_all (PAPER.md:54
 * max_pooling_2d(ksize=4, stride=str, pad=1, cover_all=True)). */
typedef struct {
  int32_t conv_type; /* LBCNN_CONV_FULL: n_kernels kernels of k x k x Cin; LBCNN_CONV_DEPTHWISE: multiplier M = n_kernels */
  int32_t n_kernels;
  int32_t ksize;     /* odd (3, 5, ...) */
  int32_t act;       /* LBCNN_ACT_NONE = the paper ("Nonlinearity achieved in Max-pool") */
  int32_t pool_k, pool_s, pool_p, pool_cover_all; /* (4,2,1,1) = paper; (2,2,0,0), (4,4,0,0) = BASELINE configs; (1,1,0,0) = none */
} lbcnn_layer_t;

typedef struct {
  int32_t in_h, in_w, in_c;
  int32_t n_layers; /* 1..3, "Up to three full convolution macro-layers" */
  lbcnn_layer_t layer[3];
  float feature_scale; /* multiplies the exact integer feature once on store; 1.0f keeps H integer-valued */
} lbcnn_arch_t;

typedef struct lbcnn_handle_s* lbcnn_handle_t;

const char* lbcnn_version(void);
const char* lbcnn_status_string(int status);

/* Create / destroy a handle bound to CUDA device `device`.  Fails with LBCNN_ERR_CUDA when no
 * such device exists (there is no CPU path), LBCNN_ERR_NOMEM when the host allocation fails.  The
 * calling thread's current device is not changed. */
int lbcnn_create(lbcnn_handle_t* h, int device);
int lbcnn_destroy(lbcnn_handle_t h);

/* Options (testing and measurement; the defaults are the product path).
 *   LBCNN_OPT_FORCE_SIMT_EXPAND  1: lbcnn_expand always takes the exact int32 SIMT kernel
 *   LBCNN_OPT_SOLVER             LBCNN_SOLVER_AUTO: lbcnn_search_candidates runs the trailing updates of the blocked factorisation on
 *                                tcgen05 (int8 digit products of the row-scaled panel: four balanced radix-256 digits, ten of the
 *                                sixteen digit products, ~2^-27 relative against 2^-24 of an fp32 factorisation) for systems of
 *                                dimension >= 1024 whose architecture cannot produce identical or negated feature maps (last layer
 *                                FULL with >= 32 taps per kernel); everything else, and lbcnn_elm_fit on data it knows nothing
 *                                about, takes the all-fp64 factorisation.  _FP64: all-fp64 everywhere.  _MIXED: tensor-core
 *                                updates whenever the system has a trailing update -- the caller vouches that the system is not
 *                                singular up to the ridge (cond * 2^-27 << 1)
 *                                Failure mode of _AUTO / _MIXED: there is no automatic retry.  On a system that IS singular up to the
 *                                ridge (a candidate whose last layer holds the same kernel twice, or nearly collinear features)
 *                                the slice error can drive a pivot non-positive: the candidate is then flagged (d_info[k] > 0,
 *                                acc -1, left out of best / worst), never returned wrong, where the all-fp64 factorisation would
 *                                have succeeded.  To tell a precision breakdown from a truly indefinite system, run the flagged
 *                                candidates again under LBCNN_SOLVER_FP64
 *   LBCNN_OPT_STREAM_ROWS        r > 0: streamed search ("limited GPU-RAM ... reduced fraction of the training
 *                                set"): the driver expands at most r samples at a time; the exact integer Gram and right-hand side
 *                                of the chunks add up (bit-identical to the unstreamed result), the test set is scored chunk by
 *                                chunk, so the features of the whole set never exist and the workspace no longer grows with
 *                                N_train / N_test.  It takes effect when the fit is the primal branch (F < N_train) with the exact
 *                                tensor-core Gram and the fused right-hand side: no bias, integer features inside the three-digit
 *                                envelope (LBCNN_H_INTEGER's bound), n_classes <= 128; otherwise the search runs resident and
 *                                lbcnn_workspace_bytes says so through its size.  The exact Gram contracts at most 43690 samples per
 *                                launch (int32 accumulators), so r > 43690 is served with chunks of 43690; N_train itself may be
 *                                larger (the paper's full 60000): only the chunk is bounded.  0 = off
 *   LBCNN_OPT_DUAL_TRICK         0: the search driver forms W = H^T Z for EVERY candidate of the dual branch and scores H_te W (default 1:
 *                                when all candidates fit one chunk, train and test features are stacked, the exact Gram of the
 *                                stack carries the cross-Gram K_te = H_te H^T, the logits K_te (H H^T + I/C)^-1 T come out of the
 *                                factorisation's appended rows, and W is formed for the best candidate only)
 *   LBCNN_OPT_MID_PANEL          width (multiple of 64; default 256; 0 = none) of the blocks inside a panel whose 64-column steps
 *                                run in fp64; a finished block updates the rest of its panel on the tensor pipe
 *   LBCNN_OPT_PANEL              panel width (multiple of 64, 64..1024; default 1024) of the blocked Cholesky when its trailing
 *                                updates run on the tensor pipe (measurement)
 *   LBCNN_OPT_DEFLATE            d = 0..64 (default 16): the first d columns of the factor -- they carry the common mode of the
 *                                all-positive features -- update the matrix beyond the first block in fp64 instead of through
 *                                the int8 slices; 0 = everything through the slices
 *   LBCNN_OPT_SCORER             LBCNN_SCORER_AUTO: the search driver scores its integer features on the tensor pipe (int8 digit
 *                                products, rows inside the error bound re-evaluated in fp64 -- the decision equals the fp64
 *                                argmax), lbcnn_elm_score uses the fp64 kernel; _FP64: fp64 everywhere; _TENSOR: lbcnn_elm_score
 *                                takes the tensor-pipe kernel too (needs lbcnn_score_workspace_bytes of workspace; rows holding
 *                                non-integer or out-of-range features are re-evaluated in fp64, so any H stays correct) */
enum { LBCNN_OPT_FORCE_SIMT_EXPAND = 0, LBCNN_OPT_SOLVER = 1, /* 2: retired (never had an effect) */ LBCNN_OPT_PANEL = 3, LBCNN_OPT_DEFLATE = 5,
       LBCNN_OPT_SCORER = 6, LBCNN_OPT_MID_PANEL = 7, LBCNN_OPT_STREAM_ROWS = 8, LBCNN_OPT_DUAL_TRICK = 9 };
enum { LBCNN_SCORER_AUTO = 0, LBCNN_SCORER_FP64 = 1, LBCNN_SCORER_TENSOR = 2 };
enum { LBCNN_SOLVER_AUTO = 0, LBCNN_SOLVER_FP64 = 1, LBCNN_SOLVER_MIXED = 2 };
int lbcnn_set_option(lbcnn_handle_t h, int option, int value);

/* Host-only shape arithmetic ("feature vector with size 15680"; Tables II-V).
 * F = Cout_last * Hout * Wout; out_hwc = {Hout, Wout, Cout} of the last layer (may be NULL). */
int lbcnn_feature_dim(const lbcnn_arch_t* arch, int64_t* F, int32_t out_hwc[3]);
/* Number of int8 weights and int32 biases in ONE candidate kernel set. */
int lbcnn_kernel_set_size(const lbcnn_arch_t* arch, int64_t* n_weights, int64_t* n_bias);

/* Workspace.  lbcnn_workspace_bytes gives the size with which lbcnn_search_candidates processes
 * min(n_cand, as many candidates as fit in `budget_bytes`) candidates per chunk (budget 0 = no cap).
 * min_bytes (may be NULL) = the size for one candidate per chunk.  `h` may be NULL (pure host arithmetic
 * for a B200).  The stand-alone calls have their own queries: lbcnn_fit_workspace_bytes for
 * lbcnn_elm_fit with the SAME flags, lbcnn_expand_workspace_bytes for lbcnn_expand.  The workspace
 * stays owned by the caller and must outlive every call enqueued with it. */
int lbcnn_workspace_bytes(lbcnn_handle_t h, const lbcnn_arch_t* arch, int64_t n_train, int64_t n_test,
                          int32_t n_classes, int32_t n_cand, size_t budget_bytes, size_t* bytes, size_t* min_bytes);
/* d_ws: 256-byte aligned, at least 256 bytes (its first 256 bytes are zeroed with a blocking cudaMemset: the
 * measurement counters of lbcnn_get_op_stats), or NULL with bytes = 0 to detach.  A configuration call, not stream-ordered:
 * do not call it while work enqueued with the previous workspace is still running. */
int lbcnn_set_workspace(lbcnn_handle_t h, void* d_ws, size_t bytes);
/* Workspace a stand-alone lbcnn_elm_fit(n, F, n_classes, n_cand, flags) needs (host-only arithmetic). */
int lbcnn_fit_workspace_bytes(int64_t n, int64_t F, int32_t n_classes, int32_t n_cand, uint32_t flags, size_t* bytes);
/* Workspace lbcnn_expand needs for n_cand candidates of this architecture: the +-1 kernel sets re-laid-out as
 * tensor-core operands (about 10 KB per candidate); 0 when the architecture takes the SIMT kernel. */
int lbcnn_expand_workspace_bytes(lbcnn_handle_t h, const lbcnn_arch_t* arch, int32_t n_cand, int32_t has_bias, size_t* bytes);

/* Expander: d_H[k][i][:] = feature_scale * flatten(layers(image i; kernel set k)).
 * The integer feature is exact (signed adds of uint8 pixels, abs < 2^24); the only rounding is the
 * one fp32 multiply by feature_scale.  d_bias may be NULL (= 0).  Scratch: the first
 * lbcnn_expand_workspace_bytes() bytes of the workspace (LBCNN_ERR_WORKSPACE when absent or too small). */
int lbcnn_expand(lbcnn_handle_t h, const lbcnn_arch_t* arch, const uint8_t* d_images /*[n][H][W][C]*/, int64_t n,
                 const int8_t* d_kernels /*[n_cand][n_weights]*/, const int32_t* d_bias /*[n_cand][n_bias] or NULL*/,
                 int32_t n_cand, float* d_H /*[n_cand][n][F]*/, void* stream);

/* Which kernel lbcnn_expand takes for this architecture (host-only; `h` supplies the device's shared-memory limit):
 * LBCNN_EXPAND_TENSOR = the tcgen05 int8 implicit-GEMM kernel (FULL convolutions, 1-2 layers, pooling with
 * k = s in {1,2,4}, p = 0, no cover_all, sizes divisible by the pool, no bias, layer-1 Cout <= 16 when a second layer
 * follows, 255 k^2 Cin <= 8191); LBCNN_EXPAND_SIMT = the exact int32 kernel that covers everything else
 * (depthwise, three layers, padded / overlapping / cover_all pooling, bias).  Both compute the same integers. */
enum { LBCNN_EXPAND_SIMT = 0, LBCNN_EXPAND_TENSOR = 1 };
int lbcnn_expand_path(lbcnn_handle_t h, const lbcnn_arch_t* arch, int32_t has_bias, int32_t* path);

/* ELM0 fit: W = argmin ||h_scale*H W - T||^2 + ||W||^2 / C with T the one-hot
 * ("categorical") coding of the labels, i.e.
 *   F <  n ("LLL"):  W = solve(I/C + H^T H, H^T T)
 *   F >= n ("MMM"):  W = H^T solve(I/C + H H^T, T)
 * on the logical features h_scale * d_H.  The Gram matrix is accumulated in fp64 (exact for
 * LBCNN_H_INTEGER data), the system is solved by a blocked fp64 Cholesky (no pivoting, no jitter)
 * and W is rounded once to fp32.  Needs the workspace.  d_info[k] = 0 or failing pivot + 1. */
int lbcnn_elm_fit(lbcnn_handle_t h, const float* d_H /*[n_cand][n][F]*/, int64_t n, int64_t F, float h_scale,
                  uint32_t flags, const int32_t* d_labels /*[n]*/, int32_t n_classes, float C, int32_t n_cand,
                  float* d_W /*[n_cand][F][n_classes]*/, int32_t* d_info /*[n_cand]*/, void* stream);

/* Score ("applied the feature vector directly to the Adaline output layer"; accuracy =
 * "fraction of correctly recognized samples in a test set"):
 *   logits = h_scale * d_H[k] . d_W[k];  pred = FIRST index of the maximum;  correct = #(pred == label).
 * d_labels, d_pred, d_correct may each be NULL.  Needs no workspace. */
int lbcnn_elm_score(lbcnn_handle_t h, const float* d_H /*[n_cand][n][F]*/, int64_t n, int64_t F, float h_scale,
                    const float* d_W /*[n_cand][F][n_classes]*/, int32_t n_classes, const int32_t* d_labels /*[n] or NULL*/,
                    int32_t n_cand, int32_t* d_pred /*[n_cand][n] or NULL*/, int32_t* d_correct /*[n_cand] or NULL*/,
                    void* stream);

/* The search loop (one trial per candidate kernel set, keep best and lowest):
 * for every candidate k: expand train and test, fit on train, score on test;
 *   d_acc[k] = correct / n_test, or -1 when the fit failed (d_info[k] != 0);
 *   d_best[0] = first k attaining the maximum accuracy, d_best[1] = first k attaining the minimum
 *   among candidates whose fit succeeded (all failed: 0, 0);
 *   d_W_best (may be NULL) = W of candidate d_best[0], acting on arch->feature_scale * integer features.
 * Candidates are processed in chunks sized by the workspace; nothing crosses to the host. */
int lbcnn_search_candidates(lbcnn_handle_t h, const lbcnn_arch_t* arch,
                            const uint8_t* d_train, const int32_t* d_train_labels, int64_t n_train,
                            const uint8_t* d_test, const int32_t* d_test_labels, int64_t n_test,
                            int32_t n_classes, float C,
                            const int8_t* d_kernels, const int32_t* d_bias /*or NULL*/, int32_t n_cand,
                            float* d_acc /*[n_cand]*/, int32_t* d_correct /*[n_cand]*/, int32_t* d_info /*[n_cand]*/,
                            int32_t* d_best /*[2]*/, float* d_W_best /*[F][n_classes] or NULL*/, void* stream);

/* The same search loop with HOST buffers: every h_* pointer is host memory (pinned memory
 * makes the copies asynchronous), layouts as in lbcnn_search_candidates.  The call stages the inputs into the
 * first lbcnn_host_staging_bytes() bytes of the workspace with cudaMemcpyAsync on `stream` (the notebook's
 * Cell 2 "move train/test to GPU memory"), runs the loop in the rest of the workspace, copies
 * acc / correct / info / best (/ W_best) back and SYNCHRONISES the stream before returning (the only
 * compute entry point that does).  Workspace needed: lbcnn_host_staging_bytes + a size
 * lbcnn_workspace_bytes accepts (>= its min_bytes); too small -> LBCNN_ERR_WORKSPACE. */
int lbcnn_host_staging_bytes(const lbcnn_arch_t* arch, int64_t n_train, int64_t n_test, int32_t n_classes,
                             int32_t n_cand, int32_t has_bias, size_t* bytes);
int lbcnn_search_candidates_host(lbcnn_handle_t h, const lbcnn_arch_t* arch,
                                 const uint8_t* h_train, const int32_t* h_train_labels, int64_t n_train,
                                 const uint8_t* h_test, const int32_t* h_test_labels, int64_t n_test,
                                 int32_t n_classes, float C,
                                 const int8_t* h_kernels, const int32_t* h_bias /*or NULL*/, int32_t n_cand,
                                 float* h_acc /*[n_cand]*/, int32_t* h_correct /*[n_cand]*/, int32_t* h_info /*[n_cand]*/,
                                 int32_t* h_best /*[2]*/, float* h_W_best /*[F][n_classes] or NULL*/, void* stream);

/* <= 8-bit fixed-point output layer ("weights represented as 8 bits integers"; Cell 12, PAPER.md:94, 98;
 * the scheme is not stated -- reading DESIGN.md R16): per candidate ONE symmetric scale,
 *   q[f][c] = clip(rint(W[f][c] * (qmax / max|W|)), -qmax, qmax),  qmax = 2^(bits-1) - 1,  2 <= bits <= 8,
 * the product taken in fp64 and rounded half to even; d_scale[k] = max|W_k| / qmax (so W ~ d_scale[k] * q).  No workspace. */
int lbcnn_quantize_output_layer(lbcnn_handle_t h, const float* d_W /*[n_cand][F][n_classes]*/, int64_t F, int32_t n_classes,
                                int32_t n_cand, int32_t bits, int8_t* d_Wq /*[n_cand][F][n_classes]*/,
                                float* d_scale /*[n_cand]*/, void* stream);
/* Score with the quantised layer: pred = argmax_c sum_f H[n][f] * q[f][c] (first index on ties); the common positive scale
 * cannot change the argmax.  For integer-valued H (the expander's output with feature_scale = 1) the logits are EXACT
 * integers (int8 digit products on the tensor pipe, int64 recombination); a row holding a non-integer or out-of-range
 * value, and exact ties, are evaluated in fp64.  Needs lbcnn_score_workspace_bytes of workspace; n_classes <= 128,
 * F a multiple of 4 and <= 43690, d_H 16-byte aligned (else LBCNN_ERR_SHAPE). */
int lbcnn_elm_score_q(lbcnn_handle_t h, const float* d_H /*[n_cand][n][F]*/, int64_t n, int64_t F,
                      const int8_t* d_Wq /*[n_cand][F][n_classes]*/, int32_t n_classes, const int32_t* d_labels /*[n] or NULL*/,
                      int32_t n_cand, int32_t* d_pred /*[n_cand][n] or NULL*/, int32_t* d_correct /*[n_cand] or NULL*/, void* stream);

/* A non-random candidate generator ("nature inspired optimization methods (such as genetic algorithms or swarm
 * intelligence methods)"; the paper gives no algorithm -- reading DESIGN.md R17): ONE generation of an elitist
 * genetic search.  From this generation's kernel sets and the accuracies lbcnn_search_candidates returned for them:
 *   1. rank the candidates by accuracy, best first, equal accuracies by index (a failed fit has accuracy -1: last);
 *   2. d_next[0 .. n_elite-1] = the n_elite best kernel sets, unchanged, in rank order;
 *   3. every other child j draws two parents, each the better-ranked of two uniformly drawn candidates (binary tournament),
 *      takes every tap from parent 1 or parent 2 with probability 1/2 (uniform crossover) and flips it with probability
 *      mut_ppm / 10^6 (mutation).
 * Random numbers: u64 draw(i) = mix(ckey + G (i + 1)), ckey = mix(key + 0xBF58476D1CE4E5B9 (j + 1)),
 * key = mix(seed XOR G (generation + 1)), G = 0x9E3779B97F4A7C15, mix = the splitmix64 finaliser; draws 0,1 / 2,3 are the
 * tournament candidates (mod n_cand), draw 4 + t decides tap t (bit 0: parent; (draw >> 20) mod 10^6 < mut_ppm: flip).
 * Byte work, bit-exact against the oracle.  Needs 8 * n_cand bytes of workspace; n_cand <= 16384; d_next != d_kernels. */
int lbcnn_evolve_candidates(lbcnn_handle_t h, const int8_t* d_kernels /*[n_cand][n_weights]*/, const float* d_acc /*[n_cand]*/,
                            int32_t n_cand, int64_t n_weights, int32_t n_elite, uint32_t mut_ppm, uint64_t seed,
                            uint32_t generation, int8_t* d_next /*[n_cand][n_weights]*/, void* stream);

/* lbcnn_evolve_candidates for callers that cannot hand the library a workspace.
 *
 * Every other compute call here takes its scratch from the buffer given to lbcnn_set_workspace, so somebody has to
 * allocate device memory first.  Some programs cannot: a plug-in that its host application hands input and output buffers
 * and nothing else; a process whose HBM was given whole to a memory pool at start-up, where a later cudaMalloc fails or
 * comes out of somebody else's budget; a control loop that must not stall, for which cudaMalloc / cudaFree are off limits
 * because they synchronise the whole device.  For them this entry point runs the same generation step (same arguments,
 * same kernels, byte-for-byte the same d_next) with NO workspace: the ranking scratch (8 bytes per candidate) lives in an
 * array compiled into the library, LBCNN_EVOLVE_STATIC_MAX_CAND * 8 bytes = 128 KB.  The handle needs no workspace; the
 * call makes no cudaMalloc / cudaFree and calls no library routine that allocates.  The caller passes inputs and outputs only.
 *
 * What that costs, and the rules that come with it:
 *   - Limit: n_cand <= LBCNN_EVOLVE_STATIC_MAX_CAND.  A larger population is refused with LBCNN_ERR_STATIC_LIMIT (nothing
 *     is enqueued); it needs lbcnn_evolve_candidates and a workspace.  All other argument rules are lbcnn_evolve_candidates'.
 *   - Footprint: the 128 KB belong to the library image, so every GPU on which this process uses liblbcnn holds them from the
 *     moment the library's code is loaded there until the process exits, whether or not this entry point is ever called.
 *   - First call on a device: the library looks the array's device address up once per device (cudaGetSymbolAddress, with
 *     that device current) and remembers it.  The look-up may make the CUDA runtime load the library's code onto the GPU,
 *     so make the first call on each device during start-up, outside any stream capture and outside the part of the program
 *     that must not stall.  Later calls on that device only enqueue work.
 *   - The handle's device must be the calling thread's current device (checked here: LBCNN_ERR_INVALID_ARG otherwise),
 *     because the address belongs to the current device.
 *   - One array per GPU, shared by every handle, stream and host thread of the process.  Each call clears the part it uses
 *     (stream-ordered, before its kernels) and then overwrites it, so nothing carries over from the previous call; but two
 *     calls whose GPU work can overlap -- different streams, or different handles on the same GPU -- write the same bytes
 *     and race.  Keep all calls of one GPU on one stream, or order them with events.  The array's contents after a call
 *     are unspecified.
 * Like the other compute calls it only enqueues on `stream` and does not synchronise. */
#define LBCNN_EVOLVE_STATIC_MAX_CAND 16384
int lbcnn_evolve_candidates_static(lbcnn_handle_t h, const int8_t* d_kernels /*[n_cand][n_weights]*/, const float* d_acc /*[n_cand]*/,
                                   int32_t n_cand, int64_t n_weights, int32_t n_elite, uint32_t mut_ppm, uint64_t seed,
                                   uint32_t generation, int8_t* d_next /*[n_cand][n_weights]*/, void* stream);

/* Gradient refinement of the output layer on the full training set (the notebook's Cell 10, "training the output
 * layer with the full dataset"; +0.73 pp on MNIST).  The paper names neither loss, optimiser nor schedule --
 * reading DESIGN.md R18 (= SPEC.md:324, 355): softmax cross-entropy; adaptive moment estimation; per mini-batch
 *   Z = h_scale H_b W,  P = softmax(Z),  G = h_scale H_b^T (P - T) / |batch|,
 *   m = b1 m + (1 - b1) G,  v = b2 v + (1 - b2) G^2,  W -= lr (m / (1 - b1^t)) / (sqrt(v / (1 - b2^t)) + eps),
 * sample j of epoch e is (a j + b) mod n with a (coprime to n) and b drawn from the counter-based generator of
 * lbcnn_evolve_candidates: a = 1 + draw(seed, e, 0, 0) mod (n - 1), advanced by a = a mod (n - 1) + 1 until gcd(a, n) = 1,
 * b = draw(seed, e, 0, 1) mod n.  The last batch of an epoch may be short.  fp64 arithmetic; d_W (fp32) is read as the
 * starting point (e.g. the ELM fit of the search on a reduced subset) and overwritten with the result; d_loss (may be NULL)
 * receives the mean cross-entropy of each epoch.  epochs = 0 leaves W unchanged.  One candidate; the binary kernels are
 * frozen by construction (the features are the input).  Needs lbcnn_refine_workspace_bytes of workspace. */
typedef struct {
  int32_t epochs;  /* >= 0 (SPEC default 10) */
  int32_t batch;   /* >= 1 (128) */
  float lr;        /* > 0 (1e-3) */
  float beta1, beta2, eps; /* 0.9, 0.999, 1e-8 */
  uint64_t seed;
} lbcnn_refine_t;
int lbcnn_refine_workspace_bytes(int64_t F, int32_t n_classes, const lbcnn_refine_t* cfg, size_t* bytes);
int lbcnn_refine_output_layer(lbcnn_handle_t h, const float* d_H /*[n][F]*/, int64_t n, int64_t F, float h_scale,
                              const int32_t* d_labels /*[n]*/, int32_t n_classes, const lbcnn_refine_t* cfg,
                              float* d_W /*[F][n_classes], in / out*/, float* d_loss /*[epochs] or NULL*/, void* stream);

/* Workspace lbcnn_elm_score needs under LBCNN_SCORER_TENSOR (host-only arithmetic; 0 is never returned). */
int lbcnn_score_workspace_bytes(int64_t n, int64_t F, int32_t n_classes, int32_t n_cand, size_t* bytes);

/* Measurement: int8 multiply-adds the tensor-core kernels have issued since the last call (or since
 * lbcnn_set_workspace), counted on the device in the first 256 bytes of the workspace (every size query above
 * includes them): h_counts[0] = the exact Gram (F1), h_counts[1] = the Cholesky trailing updates (F3).
 * Copies two words back, resets them and SYNCHRONISES the device -- call it outside timed regions. */
int lbcnn_get_op_stats(lbcnn_handle_t h, uint64_t h_counts[2]);

/* Number of kernel launches the library has enqueued through this handle since creation (for
 * bench.py's gpu_launches claim). */
int lbcnn_launch_count(lbcnn_handle_t h, int64_t* count);

/* Per-phase device timing, for measurement only (bench.py's roofline object).  With profiling on,
 * every phase the library enqueues is bracketed by a pair of CUDA events on the caller's stream.
 * lbcnn_get_phase_times BLOCKS until the recorded events have completed (the one call of this
 * library that synchronises), adds the elapsed milliseconds and launch-bracket counts per phase
 * into h_ms / h_count (host arrays of LBCNN_N_PHASES entries, overwritten) and clears the record. */
enum { LBCNN_PHASE_EXPAND = 0, LBCNN_PHASE_GRAM = 1, LBCNN_PHASE_RHS = 2, LBCNN_PHASE_SOLVE = 3,
       LBCNN_PHASE_SCORE = 4, LBCNN_PHASE_FINISH = 5, LBCNN_N_PHASES = 6 };
int lbcnn_set_profiling(lbcnn_handle_t h, int enable);
int lbcnn_get_phase_times(lbcnn_handle_t h, float* h_ms, int32_t* h_count);

#ifdef __cplusplus
}
#endif
#endif /* LBCNN_H_ */
