/*
 * lbcnn_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU implementation of what the LB-CNN kernel-selection
 * inner loop computes (arXiv 2106.15350), written from the paper's definitions.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 * It shares no code, header, table or helper with the CUDA path (paper_2106_15350_b200/csrc).
 *
 * Arithmetic: the expander is integer (int64 accumulators): the kernels are +-1 and the pixels
 * are uint8, so every intermediate is an exact integer.  The ELM fit and the score are fp64
 * ("Q16": the paper does not state a precision).  There is no blocking, fusion or reordering
 * beyond the definitions; OpenMP only distributes independent outputs (samples, matrix rows)
 * over threads and `omp simd reduction` lets the compiler vectorise one dot product.
 *
 * Parity pins (tests/test_oracle_pins.py): paper-printed feature sizes / parameter bits
 * (Tables II-V), brute-force convolution and pooling in Python, worked examples
 * in tests/golden/, normal-equation residual, pseudo-inverse limit, primal == dual, sign flip.
 * Unpinned: nothing in this file (accuracies / timings printed in the paper need its datasets and
 * are not used at all).
 *
 * Passages followed:
 *   conv macro-layer   PAPER.md:51-55  (section II listing, lines 27-31: convolution pad=1,
 *                                       max_pooling_2d(ksize=4, stride=str, pad=1, cover_all=True))
 *   up to 3 layers + flatten
 *   depth-wise vs normal convolution
 *   ELM0 fit (both branches)            PAPER.md:61-70 of the listing = PAPER.md:64-74
 *   predict = Adaline output, argmax    PAPER.md:59; accuracy PAPER.md:23
 * Readings where the paper is silent are DESIGN.md "Readings" R1..R14 (binary alphabet +-1,
 * cross-correlation, zero conv padding (k-1)/2, -inf pool padding, CHW flatten, one-hot targets,
 * Cholesky instead of the listing's LU `solve`, ties -> lowest index).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
  int32_t conv_type; /* 0 FULL: n_kernels kernels of k x k x Cin; 1 DEPTHWISE: multiplier M, Cout = Cin*M */
  int32_t n_kernels;
  int32_t ksize;     /* odd; zero padding (ksize-1)/2, stride 1 */
  int32_t act;       /* 0 none ("Nonlinearity achieved in Max-pool"), 1 relu */
  int32_t pool_k, pool_s, pool_p, pool_cover_all;
} orc_layer;

typedef struct {
  int32_t in_h, in_w, in_c;
  int32_t n_layers;  /* 1..3 */
  orc_layer layer[3];
} orc_arch;

/* Output size of one pooling axis.  Without cover_all: floor((n+2p-k)/s)+1; with cover_all
 * (PAPER.md:54): ceil((n+2p-k)/s)+1, i.e. a final partial window is emitted.  Returns -1 if the
 * size is < 1 or some window would hold no real cell. */
int orc_pool_out_size(int n, int k, int s, int p, int cover_all) {
  if (n < 1 || k < 1 || s < 1 || p < 0) return -1;
  int span = n + 2 * p - k;
  if (span < 0) return -1;
  int out = cover_all ? (span + s - 1) / s + 1 : span / s + 1;
  if (out < 1) return -1;
  /* every window [i*s-p, i*s-p+k) must contain a real cell in [0,n) */
  for (int i = 0; i < out; ++i) {
    int lo = i * s - p, hi = lo + k; /* exclusive */
    if (lo < 0) lo = 0;
    if (hi > n) hi = n;
    if (hi <= lo) return -1;
  }
  return out;
}

/* Shape chain of the expander; F = C_out * H_out * W_out of the last layer. */
int orc_feature_dim(const orc_arch* a, int64_t* F, int32_t out_hwc[3]) {
  if (!a || a->n_layers < 1 || a->n_layers > 3 || a->in_h < 1 || a->in_w < 1 || a->in_c < 1) return 2;
  int h = a->in_h, w = a->in_w, c = a->in_c;
  for (int l = 0; l < a->n_layers; ++l) {
    const orc_layer* L = &a->layer[l];
    if (L->n_kernels < 1 || L->ksize < 1 || (L->ksize % 2) == 0) return 2;
    c = (L->conv_type == 0) ? L->n_kernels : c * L->n_kernels;
    h = orc_pool_out_size(h, L->pool_k, L->pool_s, L->pool_p, L->pool_cover_all);
    w = orc_pool_out_size(w, L->pool_k, L->pool_s, L->pool_p, L->pool_cover_all);
    if (h < 1 || w < 1) return 2;
  }
  if (F) *F = (int64_t)c * h * w;
  if (out_hwc) { out_hwc[0] = h; out_hwc[1] = w; out_hwc[2] = c; }
  return 0;
}

/* "Params (k-bits) Conv+ELM" of Tables II-V: one bit per binary weight (biases not counted),
 * 8 bits per output-layer weight ("weights represented as 8 bits integers"). */
int orc_param_bits(const orc_arch* a, int n_classes, int64_t* conv_bits, int64_t* elm_bits) {
  int64_t F; int32_t hwc[3];
  int rc = orc_feature_dim(a, &F, hwc);
  if (rc) return rc;
  int64_t bits = 0; int c = a->in_c;
  for (int l = 0; l < a->n_layers; ++l) {
    const orc_layer* L = &a->layer[l];
    bits += (int64_t)L->n_kernels * c * L->ksize * L->ksize;
    c = (L->conv_type == 0) ? L->n_kernels : c * L->n_kernels;
  }
  *conv_bits = bits; *elm_bits = F * n_classes * 8;
  return 0;
}

/* One binary convolution on one image, channels-last, cross-correlation, zero
 * padding p=(k-1)/2, stride 1 (PAPER.md:53 pad=1 for 3x3):
 *   FULL:      z[y,x,o]     = b[o]     + sum_{c,dy,dx} w[o,c,dy,dx]   * a[y+dy-p, x+dx-p, c]
 *   DEPTHWISE: z[y,x,c*M+m] = b[c*M+m] + sum_{dy,dx}   w[m,c,dy,dx]   * a[y+dy-p, x+dx-p, c]
 * w is [n_kernels][Cin][k][k] in both cases, entries +-1. */
static void conv_one(int conv_type, int nk, int k, const int64_t* a, int h, int w, int cin,
                     const int8_t* wt, const int32_t* bias, int64_t* z) {
  int p = (k - 1) / 2;
  int cout = conv_type == 0 ? nk : cin * nk;
  for (int y = 0; y < h; ++y)
    for (int x = 0; x < w; ++x)
      for (int o = 0; o < cout; ++o) {
        int64_t acc = bias ? bias[o] : 0;
        if (conv_type == 0) {
          for (int c = 0; c < cin; ++c)
            for (int dy = 0; dy < k; ++dy)
              for (int dx = 0; dx < k; ++dx) {
                int yy = y + dy - p, xx = x + dx - p;
                if (yy < 0 || yy >= h || xx < 0 || xx >= w) continue; /* zero outside */
                acc += (int64_t)wt[((o * cin + c) * k + dy) * k + dx] * a[(yy * w + xx) * cin + c];
              }
        } else {
          int c = o / nk, m = o % nk;
          for (int dy = 0; dy < k; ++dy)
            for (int dx = 0; dx < k; ++dx) {
              int yy = y + dy - p, xx = x + dx - p;
              if (yy < 0 || yy >= h || xx < 0 || xx >= w) continue;
              acc += (int64_t)wt[((m * cin + c) * k + dy) * k + dx] * a[(yy * w + xx) * cin + c];
            }
        }
        z[(y * w + x) * cout + o] = acc;
      }
}

/* Max-pool on one image: window rows i*s-p .. i*s-p+k-1 (same for columns); padding cells are
 * -inf, i.e. only in-image cells compete (R5). */
static void pool_one(const int64_t* z, int h, int w, int c, int k, int s, int p, int ho, int wo, int64_t* u) {
  for (int i = 0; i < ho; ++i)
    for (int j = 0; j < wo; ++j)
      for (int o = 0; o < c; ++o) {
        int have = 0; int64_t best = 0;
        for (int dy = 0; dy < k; ++dy)
          for (int dx = 0; dx < k; ++dx) {
            int yy = i * s - p + dy, xx = j * s - p + dx;
            if (yy < 0 || yy >= h || xx < 0 || xx >= w) continue;
            int64_t v = z[(yy * w + xx) * c + o];
            if (!have || v > best) { best = v; have = 1; }
          }
        u[(i * wo + j) * c + o] = best;
      }
}

/* Stand-alone layer pieces on a batch, for the pins (int64 in, int64 out, NHWC). */
int orc_conv(int conv_type, int n_kernels, int ksize, const int64_t* a, int64_t n, int h, int w, int cin,
             const int8_t* wt, const int32_t* bias, int64_t* z) {
  if (ksize < 1 || ksize % 2 == 0 || n_kernels < 1) return 2;
  int cout = conv_type == 0 ? n_kernels : cin * n_kernels;
  for (int64_t i = 0; i < n; ++i)
    conv_one(conv_type, n_kernels, ksize, a + i * h * w * cin, h, w, cin, wt, bias, z + i * h * w * cout);
  return 0;
}

int orc_maxpool(const int64_t* z, int64_t n, int h, int w, int c, int k, int s, int p, int cover_all, int64_t* u) {
  int ho = orc_pool_out_size(h, k, s, p, cover_all), wo = orc_pool_out_size(w, k, s, p, cover_all);
  if (ho < 1 || wo < 1) return 2;
  for (int64_t i = 0; i < n; ++i)
    pool_one(z + i * h * w * c, h, w, c, k, s, p, ho, wo, u + i * ho * wo * c);
  return 0;
}

/* Expander for ONE candidate kernel set: up to three (conv -> act -> pool) macro-layers then a
 * flatten in C,H,W order, f = (o*Hout + i)*Wout + j (R7).
 * kernels: layers concatenated, layer l = [n_kernels][Cin_l][k][k] int8 +-1.
 * bias: layers concatenated, layer l = [Cout_l] int32, or NULL = 0.
 * u: [n][F] int64, the exact integer features (before any feature_scale). */
int orc_expand(const orc_arch* a, const uint8_t* images, int64_t n, const int8_t* kernels, const int32_t* bias,
               int64_t* u) {
  int64_t F; int32_t hwc[3];
  int rc = orc_feature_dim(a, &F, hwc);
  if (rc) return rc;
  /* largest intermediate sizes */
  int64_t max_act = (int64_t)a->in_h * a->in_w * a->in_c, max_z = 0;
  {
    int h = a->in_h, w = a->in_w, c = a->in_c;
    for (int l = 0; l < a->n_layers; ++l) {
      const orc_layer* L = &a->layer[l];
      int co = L->conv_type == 0 ? L->n_kernels : c * L->n_kernels;
      if ((int64_t)h * w * co > max_z) max_z = (int64_t)h * w * co;
      h = orc_pool_out_size(h, L->pool_k, L->pool_s, L->pool_p, L->pool_cover_all);
      w = orc_pool_out_size(w, L->pool_k, L->pool_s, L->pool_p, L->pool_cover_all);
      c = co;
      if ((int64_t)h * w * c > max_act) max_act = (int64_t)h * w * c;
    }
  }
  int err = 0;
#pragma omp parallel
  {
    int64_t* act = (int64_t*)malloc(sizeof(int64_t) * max_act);
    int64_t* nxt = (int64_t*)malloc(sizeof(int64_t) * max_act);
    int64_t* z = (int64_t*)malloc(sizeof(int64_t) * max_z);
    if (!act || !nxt || !z) {
#pragma omp atomic write
      err = 1;
    } else {
#pragma omp for schedule(static)
      for (int64_t i = 0; i < n; ++i) {
        int h = a->in_h, w = a->in_w, c = a->in_c;
        const uint8_t* img = images + i * h * w * c;
        for (int64_t t = 0; t < (int64_t)h * w * c; ++t) act[t] = img[t];
        const int8_t* wt = kernels; const int32_t* bs = bias;
        for (int l = 0; l < a->n_layers; ++l) {
          const orc_layer* L = &a->layer[l];
          int co = L->conv_type == 0 ? L->n_kernels : c * L->n_kernels;
          conv_one(L->conv_type, L->n_kernels, L->ksize, act, h, w, c, wt, bs, z);
          if (L->act == 1)
            for (int64_t t = 0; t < (int64_t)h * w * co; ++t) if (z[t] < 0) z[t] = 0;
          int ho = orc_pool_out_size(h, L->pool_k, L->pool_s, L->pool_p, L->pool_cover_all);
          int wo = orc_pool_out_size(w, L->pool_k, L->pool_s, L->pool_p, L->pool_cover_all);
          pool_one(z, h, w, co, L->pool_k, L->pool_s, L->pool_p, ho, wo, nxt);
          wt += (int64_t)L->n_kernels * c * L->ksize * L->ksize;
          if (bs) bs += co;
          h = ho; w = wo; c = co;
          int64_t* tmp = act; act = nxt; nxt = tmp;
        }
        /* flatten HWC -> CHW */
        for (int o = 0; o < c; ++o)
          for (int y = 0; y < h; ++y)
            for (int x = 0; x < w; ++x)
              u[i * F + ((int64_t)o * h + y) * w + x] = act[(y * w + x) * c + o];
      }
    }
    free(act); free(nxt); free(z);
  }
  return err ? 5 : 0;
}

/* ------------------------------------------------------------------------------------------ */
/* ELM0 fit.  In this file H is samples x features (row n = feature vector of
 * sample n), the transpose of the listing's H (features x samples), so the listing's
 * H.H^T is H^T H here and H^T.H is H H^T (R9).                                         */

static double dot(const double* x, const double* y, int64_t n) {
  double s = 0.0;
#pragma omp simd reduction(+ : s)
  for (int64_t i = 0; i < n; ++i) s += x[i] * y[i];
  return s;
}

/* In-place Cholesky A = L L^T of the lower triangle (row-major, leading dimension d), no
 * pivoting, no jitter.  Returns 0, or j+1 if pivot j is not positive (LAPACK convention).
 * Cholesky-Crout: column j from the rows of L already known. */
static int cholesky(double* A, int64_t d) {
  for (int64_t j = 0; j < d; ++j) {
    double piv = A[j * d + j] - dot(A + j * d, A + j * d, j);
    if (!(piv > 0.0)) return (int)(j + 1);
    double ljj = sqrt(piv);
    A[j * d + j] = ljj;
#pragma omp parallel for schedule(static)
    for (int64_t i = j + 1; i < d; ++i)
      A[i * d + j] = (A[i * d + j] - dot(A + i * d, A + j * d, j)) / ljj;
  }
  return 0;
}

/* Solve L L^T X = B in place, B is d x m row-major. */
static void chol_solve(const double* L, int64_t d, double* B, int64_t m) {
  for (int64_t i = 0; i < d; ++i)            /* forward: L Y = B */
    for (int64_t c = 0; c < m; ++c) {
      double s = B[i * m + c];
      for (int64_t k = 0; k < i; ++k) s -= L[i * d + k] * B[k * m + c];
      B[i * m + c] = s / L[i * d + i];
    }
  for (int64_t i = d - 1; i >= 0; --i)       /* backward: L^T X = Y */
    for (int64_t c = 0; c < m; ++c) {
      double s = B[i * m + c];
      for (int64_t k = i + 1; k < d; ++k) s -= L[k * d + i] * B[k * m + c];
      B[i * m + c] = s / L[i * d + i];
    }
}

/* H: [n][F] fp64; labels in [0, classes); T[n][c] = 1 if labels[n]==c else 0 ("categorical
 * format").  force_branch: 0 = the listing's rule (F < n -> primal 'LLL', else dual
 * 'MMM'), 1 = primal, 2 = dual.  W: [F][classes].  *branch_out: 1 primal, 2 dual.
 * Returns 0, >0 = Cholesky pivot index + 1, <0 = bad argument / out of memory. */
int orc_elm_fit(const double* H, int64_t n, int64_t F, const int32_t* labels, int32_t classes, double C,
                int force_branch, double* W, int32_t* branch_out) {
  if (!H || !labels || !W || n < 1 || F < 1 || classes < 2 || !(C > 0.0)) return -1;
  for (int64_t i = 0; i < n; ++i) if (labels[i] < 0 || labels[i] >= classes) return -1;
  int primal = force_branch ? (force_branch == 1) : (F < n);
  if (branch_out) *branch_out = primal ? 1 : 2;
  int info = 0;
  if (primal) {
    /* outW = solve(I/C + H^T H, H^T T) */
    double* Ht = (double*)malloc(sizeof(double) * F * n);
    double* A = (double*)malloc(sizeof(double) * F * F);
    if (!Ht || !A) { free(Ht); free(A); return -2; }
#pragma omp parallel for schedule(static)
    for (int64_t f = 0; f < F; ++f)
      for (int64_t i = 0; i < n; ++i) Ht[f * n + i] = H[i * F + f];
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = 0; i < F; ++i)
      for (int64_t j = 0; j <= i; ++j) {
        double g = dot(Ht + i * n, Ht + j * n, n);
        if (i == j) g += 1.0 / C;
        A[i * F + j] = g; A[j * F + i] = g;
      }
    for (int64_t t = 0; t < F * classes; ++t) W[t] = 0.0;
#pragma omp parallel for schedule(static)
    for (int64_t f = 0; f < F; ++f)
      for (int64_t i = 0; i < n; ++i) W[f * classes + labels[i]] += Ht[f * n + i];   /* B = H^T T */
    info = cholesky(A, F);
    if (!info) chol_solve(A, F, W, classes);
    free(Ht); free(A);
  } else {
    /* outW = H^T solve(I/C + H H^T, T) */
    double* A = (double*)malloc(sizeof(double) * n * n);
    double* Z = (double*)calloc((size_t)n * classes, sizeof(double));
    if (!A || !Z) { free(A); free(Z); return -2; }
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = 0; i < n; ++i)
      for (int64_t j = 0; j <= i; ++j) {
        double g = dot(H + i * F, H + j * F, F);
        if (i == j) g += 1.0 / C;
        A[i * n + j] = g; A[j * n + i] = g;
      }
    for (int64_t i = 0; i < n; ++i) Z[i * classes + labels[i]] = 1.0;
    info = cholesky(A, n);
    if (!info) {
      chol_solve(A, n, Z, classes);
#pragma omp parallel for schedule(static)
      for (int64_t f = 0; f < F; ++f)
        for (int c = 0; c < classes; ++c) {
          double s = 0.0;
          for (int64_t i = 0; i < n; ++i) s += H[i * F + f] * Z[i * classes + c];
          W[f * classes + c] = s;
        }
    }
    free(A); free(Z);
  }
  return info;
}

/* Predict + accuracy count ("applied the feature vector directly to the Adaline
 * output layer"; PAPER.md:23 accuracy = fraction of correctly recognised test samples).
 * logits[n][c] = sum_f H[n][f] W[f][c]; pred = FIRST index of the maximum (R12).
 * margin (optional): top-1 minus top-2 logit, to diagnose near-ties. */
int orc_elm_score(const double* H, int64_t n, int64_t F, const double* W, int32_t classes, const int32_t* labels,
                  int32_t* pred, int64_t* correct, double* margin) {
  if (!H || !W || n < 1 || F < 1 || classes < 2) return -1;
  int64_t ok = 0;
#pragma omp parallel for schedule(static) reduction(+ : ok)
  for (int64_t i = 0; i < n; ++i) {
    int best = 0; double bv = 0.0, second = -INFINITY;
    for (int c = 0; c < classes; ++c) {
      double s = 0.0;
      for (int64_t f = 0; f < F; ++f) s += H[i * F + f] * W[f * classes + c];
      if (c == 0) { bv = s; }
      else if (s > bv) { second = bv; bv = s; best = c; }
      else if (s > second) { second = s; }
    }
    if (pred) pred[i] = best;
    if (margin) margin[i] = bv - second;
    if (labels && labels[i] == best) ok += 1;
  }
  if (correct) *correct = ok;
  return 0;
}
