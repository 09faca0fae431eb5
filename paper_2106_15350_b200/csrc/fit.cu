// fit.cu -- ELM0 fit: Gram + ridge (F1), right-hand side (F2), SPD solve (F3).
//
// System solved per candidate, on the STORED features U (logical feature = s*U, s = h_scale):
//   primal (F < n):  (U^T U + lam I) W' = U^T T,        W = W'/s
//   dual  (F >= n):  (U U^T + lam I) Z  = T,  W' = U^T Z, W = W'/s        lam = 1/(C s^2)
// which is the paper's (H^T H + I/C) W = H^T T with H = s*U divided through by s^2.
// Storage: per candidate a (dim + c) x dim fp64 matrix, row-major, leading dimension dim: the lower
// triangle of rows 0..dim-1 holds the system matrix, rows dim..dim+c-1 hold the right-hand sides
// TRANSPOSED (row = class).  A right-looking blocked Cholesky over all dim + c rows then leaves
// L in the triangle and Y^T = (L^-1 B)^T in the appended rows (forward substitution for free);
// a blocked backward sweep turns Y^T into X^T.
#include "internal.h"
#include "gemm_launch.cuh"

namespace {

constexpr int NB = 64;   // Cholesky block size

// ---------------------------------------------------------------------------------------------
// labels -> stable class-sorted sample permutation (one thread per class; deterministic)
__global__ void label_perm_kernel(const int32_t* __restrict__ y, int n, int c, int32_t* __restrict__ perm,
                                  int32_t* __restrict__ off) {
  extern __shared__ int cnt[];
  for (int t = threadIdx.x; t <= c; t += blockDim.x) cnt[t] = 0;
  __syncthreads();
  // a label outside [0, c) belongs to no class: its sample contributes an all-zero target row (include/lbcnn.h)
  for (int i = threadIdx.x; i < n; i += blockDim.x)
    if ((unsigned)y[i] < (unsigned)c) atomicAdd(&cnt[y[i] + 1], 1);
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int t = 1; t <= c; ++t) cnt[t] += cnt[t - 1];
  }
  __syncthreads();
  for (int t = threadIdx.x; t <= c; t += blockDim.x) off[t] = cnt[t];
  for (int cls = threadIdx.x; cls < c; cls += blockDim.x) {
    int w = cnt[cls];
    for (int i = 0; i < n; ++i)
      if (y[i] == cls) perm[w++] = i;
  }
}

// primal right-hand side (F2): Bt[cls][f] = sum_{n: y_n = cls} U[n][f]  (T one-hot)
__global__ void __launch_bounds__(128) rhs_primal_kernel(const float* __restrict__ U, long long n, long long F,
                                                         const int32_t* __restrict__ perm,
                                                         const int32_t* __restrict__ off, double* __restrict__ A,
                                                         long long a_stride, long long dim) {
  const long long f = (long long)blockIdx.x * 128 + threadIdx.x;
  const int cls = blockIdx.y;
  const long long z = blockIdx.z;
  if (f >= F) return;
  const float* Uz = U + z * n * F + f;
  const int lo = off[cls], hi = off[cls + 1];
  // eight independent row loads in flight per thread (the rows of one class are scattered over the sample axis)
  double s0 = 0, s1 = 0, s2 = 0, s3 = 0;
  int i = lo;
  for (; i + 7 < hi; i += 8) {
    float v[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) v[q] = __ldcs(Uz + (long long)perm[i + q] * F);
    s0 += (double)v[0] + (double)v[4]; s1 += (double)v[1] + (double)v[5];
    s2 += (double)v[2] + (double)v[6]; s3 += (double)v[3] + (double)v[7];
  }
  for (; i < hi; ++i) s0 += Uz[(long long)perm[i] * F];
  A[z * a_stride + (dim + cls) * dim + f] = (s0 + s1) + (s2 + s3);
}

// dual right-hand side: rows dim.. = T^T (c x n one-hot)
__global__ void rhs_dual_kernel(const int32_t* __restrict__ y, long long n, int c, double* __restrict__ A,
                                long long a_stride) {
  const long long z = blockIdx.z;
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n * c) return;
  const int cls = (int)(t / n);
  const long long i = t % n;
  A[z * a_stride + (n + cls) * n + i] = (y[i] == cls) ? 1.0 : 0.0;
}

// ---------------------------------------------------------------------------------------------
// blocked Cholesky pieces (F3).  Matrix of candidate z at A + z*a_stride, leading dimension ld = dim.

// factorise the nbj x nbj diagonal block at (j0, j0); a non-positive pivot records info = index + 1
// (first failure wins) and continues with pivot 1 so that the candidate's data stays finite.
// Also writes Linv = L11^-1 (nbj x nbj, lower triangular, zeros above the diagonal, pitch NB) to
// linv + blockIdx.x * linv_stride: the panel solve and the backward sweep then are plain products.
__global__ void __launch_bounds__(256) potrf_diag_kernel(double* __restrict__ A, long long a_stride, long long ld,
                                                         int j0, int nbj, int32_t* __restrict__ info,
                                                         double* __restrict__ linv, long long linv_stride) {
  extern __shared__ double potrf_sh[];
  double (*S)[NB + 1] = reinterpret_cast<double (*)[NB + 1]>(potrf_sh);
  double (*X)[NB + 1] = reinterpret_cast<double (*)[NB + 1]>(potrf_sh + NB * (NB + 1));
  double* Az = A + blockIdx.x * a_stride + (long long)j0 * ld + j0;
  // Right-looking factorisation with the block in REGISTERS: thread (ty, tx) of a 16 x 16 grid owns the 4 x 4
  // elements (ty + 16 a, tx + 16 b).  Per column j: its owners publish the current column, one barrier, then every
  // thread scales and applies the rank-1 update to its own elements (no integer division, one barrier per column).
  __shared__ double colraw[2][NB];
  const int ty = threadIdx.x >> 4, tx = threadIdx.x & 15;
  double r[4][4];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      const int i = ty + 16 * a, c = tx + 16 * b;
      r[a][b] = (i < nbj && c <= i) ? Az[(long long)i * ld + c] : ((i == c) ? 1.0 : 0.0);   // identity padding
    }
#pragma unroll
  for (int jb = 0; jb < 4; ++jb) {                 // block column of the 16 x 16 thread grid: static register indices
    for (int jj = 0; jj < 16; ++jj) {
      const int j = jb * 16 + jj;
      if (j >= nbj) break;
      double* col = colraw[j & 1];
      if (tx == jj) {
#pragma unroll
        for (int a = 0; a < 4; ++a) col[ty + 16 * a] = r[a][jb];
      }
      __syncthreads();
      double piv = col[j];
      if (!(piv > 0.0)) {
        if (threadIdx.x == 0 && info[blockIdx.x] == 0) info[blockIdx.x] = j0 + j + 1;
        piv = 1.0;
      }
      const double inv = rsqrt(piv);               // 1 / l
      const double l = piv * inv;
      double li[4], lc[4];
#pragma unroll
      for (int a = 0; a < 4; ++a) li[a] = col[ty + 16 * a] * inv;
#pragma unroll
      for (int b = 0; b < 4; ++b) lc[b] = col[tx + 16 * b] * inv;
#pragma unroll
      for (int a = 0; a < 4; ++a) {
        const int i = ty + 16 * a;
        if (tx == jj) r[a][jb] = (i == j) ? l : ((i > j) ? li[a] : r[a][jb]);
        else if (tx > jj && tx + 16 * jb <= i) r[a][jb] = fma(-li[a], lc[jb], r[a][jb]);
#pragma unroll
        for (int b = 0; b < 4; ++b)
          if (b > jb && tx + 16 * b <= i) r[a][b] = fma(-li[a], lc[b], r[a][b]);
      }
    }
  }
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      const int i = ty + 16 * a, c = tx + 16 * b;
      S[i][c] = r[a][b];
      if (i < nbj && c <= i) Az[(long long)i * ld + c] = r[a][b];
    }
  __syncthreads();
  // inverse of the triangular factor by forward substitution (L X = I): four adjacent lanes share a column and split
  // the inner sum, so a warp advances eight columns with two shuffles per row
  {
    const int c = threadIdx.x >> 2, part = threadIdx.x & 3;
    const int c_min = (threadIdx.x >> 5) * 8;        // first column of this warp
    if (part == 0) {
      for (int i = 0; i < c; ++i) X[i][c] = 0.0;
      X[c][c] = 1.0 / S[c][c];
    }
    __syncwarp();
    for (int i = c_min + 1; i < nbj; ++i) {
      double acc = 0.0;
      if (i > c)
        for (int k = c + part; k < i; k += 4) acc = fma(S[i][k], X[k][c], acc);
      acc += __shfl_xor_sync(0xffffffffu, acc, 1);
      acc += __shfl_xor_sync(0xffffffffu, acc, 2);
      if (part == 0 && i > c) X[i][c] = -acc / S[i][i];
      __syncwarp();
    }
  }
  __syncthreads();
  double* Lz = linv + blockIdx.x * linv_stride;
  for (int e = threadIdx.x; e < NB * NB; e += blockDim.x) {
    const int i = e / NB, c = e % NB;
    Lz[e] = (i < nbj && c < nbj) ? X[i][c] : 0.0;
  }
}

// primal: W[f][cls] = X^T[cls][f] / s, rounded once to fp32
__global__ void w_from_xt_kernel(const double* __restrict__ A, long long a_stride, long long dim, int c, double inv_s,
                                 float* __restrict__ W) {
  const long long z = blockIdx.z;
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= dim * c) return;
  const long long f = t / c;
  const int cls = (int)(t % c);
  W[z * dim * c + t] = (float)(A[z * a_stride + (dim + cls) * dim + f] * inv_s);
}

// dual branch, kernel trick: class = first maximum of a row of logits [n_te][c] (fp64); one warp per 32 rows
__global__ void __launch_bounds__(256) dual_argmax_kernel(const double* __restrict__ logits, long long n_te, int c,
                                                          const int32_t* __restrict__ y, int32_t* __restrict__ correct) {
  const long long z = blockIdx.y;
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  int ok = 0;
  if (i < n_te) {
    const double* l = logits + (z * n_te + i) * c;
    double best = l[0]; int bi = 0;
    for (int j = 1; j < c; ++j) { const double v = l[j]; if (v > best) { best = v; bi = j; } }
    ok = (y[i] == bi) ? 1 : 0;
  }
  ok = __reduce_add_sync(0xffffffffu, ok);
  if ((threadIdx.x & 31) == 0 && ok) atomicAdd(&correct[z], ok);
}

// W of the best candidate only (its index is read on the device): W[f][cls] = (1/s) sum_n U[n][f] Z^T[cls][n]
__global__ void __launch_bounds__(128) w_best_dual_kernel(const int32_t* __restrict__ best, const float* __restrict__ Hall,
                                                          long long n, long long n_rows, long long F, const double* __restrict__ A,
                                                          long long a_stride, long long ld, long long dim, int c, double inv_s,
                                                          float* __restrict__ W) {
  const long long z = best[0];
  const long long f = (long long)blockIdx.x * 128 + threadIdx.x;
  const int c0 = blockIdx.y * 8;
  if (f >= F) return;
  const float* U = Hall + z * n_rows * F + f;
  const double* Zt = A + z * a_stride + (dim + c0) * ld;
  double acc[8];
#pragma unroll
  for (int q = 0; q < 8; ++q) acc[q] = 0.0;
  const int nc = (c - c0 < 8) ? c - c0 : 8;
  for (long long i = 0; i < n; ++i) {
    const double u = (double)U[i * F];
#pragma unroll
    for (int q = 0; q < 8; ++q)
      if (q < nc) acc[q] = fma(u, Zt[q * ld + i], acc[q]);
  }
#pragma unroll
  for (int q = 0; q < 8; ++q)
    if (q < nc) W[f * c + c0 + q] = (float)(acc[q] * inv_s);
}

}  // namespace

int lb_launch_w_best_dual(lbcnn_handle_s* h, void* ws, const FitPlan& pl, const int32_t* d_best, const float* d_Hall, int64_t n,
                          int64_t F, float h_scale, int n_classes, float* d_W_best, cudaStream_t st) {
  double* A = reinterpret_cast<double*>(reinterpret_cast<char*>(ws) + pl.a_off);
  dim3 grid((unsigned)((F + 127) / 128), (unsigned)((n_classes + 7) / 8));
  w_best_dual_kernel<<<grid, 128, 0, st>>>(d_best, d_Hall, n, n + pl.n_extra, F, A, pl.rows * pl.dim, pl.dim, pl.dim, n_classes,
                                           1.0 / (double)h_scale, d_W_best);
  h->launches += 1;
  LB_CUDA_OK(cudaGetLastError());
  return LBCNN_OK;
}

// ---------------------------------------------------------------------------------------------
void lb_fit_plan(int64_t n, int64_t F, int n_classes, int n_cand, uint32_t flags, FitPlan* p, int64_t n_ws, int64_t n_extra) {
  if (n_ws <= 0 || n_ws > n) n_ws = n;
  int primal = (F < n) ? 1 : 0;                       // PAPER.md:68 `if n_inputs<Ntr` ('LLL'), else 'MMM'
  if (flags & LBCNN_FORCE_PRIMAL) primal = 1;
  if (flags & LBCNN_FORCE_DUAL) primal = 0;
  p->primal = primal;
  p->dim = primal ? F : n;
  // the int32 bound of the exact Gram is on the samples contracted per LAUNCH: a streamed plan (n_ws < n) adds the exact
  // fp64 Grams of chunks of n_ws rows, so its bound is on n_ws, not on n (N = 60000 streams in chunks of <= 43690)
  p->use_tc = ((flags & LBCNN_H_INTEGER) && lb_gram_tc_usable(primal ? n_ws : n, F, primal != 0)) ? 1 : 0;
  p->n_extra = (!primal && p->use_tc && n_extra > 0) ? n_extra : 0;
  p->rows = p->dim + n_classes + p->n_extra;
  p->a_bytes = (size_t)p->rows * (size_t)p->dim * sizeof(double);
  size_t off = 0;
  p->perm_off = off; off += (size_t)lb_align_up(n * 4, 256);
  p->off_off = off;  off += (size_t)lb_align_up(((int64_t)n_classes + 1) * 4, 256);
  p->a_off = off;    off += (size_t)lb_align_up((int64_t)p->a_bytes * n_cand, 256);
  p->tc_off = off;   p->fuse_rhs = (p->use_tc && primal && lb_gram_tc_fuse_rhs(F, n_classes)) ? 1 : 0;
  if (p->use_tc) off += lb_gram_tc_ws_bytes(n_ws + p->n_extra, F, n_cand, p->fuse_rhs ? n_classes : 0);
  p->lg_off = off;   off += (size_t)lb_align_up((int64_t)n_cand * p->n_extra * n_classes * 8, 256);
  p->linv_off = off; off += (size_t)lb_align_up((int64_t)n_cand * ((p->dim + NB - 1) / NB) * NB * NB * 8, 256);
  // digit planes + row scales of the tensor-core trailing updates (chol_tc.cu), for systems large enough to have them
  p->allow_tc = 0;
  p->stc_kmax = (p->dim >= LB_STC_MIN_DIM) ? LB_STC_KMAX : 0;
  p->stc_off = off;
  if (p->stc_kmax) off += lb_chol_tc_ws_bytes(p->rows, n_cand, p->stc_kmax);
  p->total = off;
}

int lb_launch_fit(lbcnn_handle_s* h, void* ws, const FitPlan& pl, const float* d_H, int64_t n, int64_t F, float h_scale,
                  const int32_t* d_labels, int n_classes, float C, int n_cand, float* d_W, int32_t* d_info,
                  cudaStream_t st, const FitStream* fs, const DualScore* ds) {
  char* base = reinterpret_cast<char*>(ws);
  int32_t* perm = reinterpret_cast<int32_t*>(base + pl.perm_off);
  int32_t* off = reinterpret_cast<int32_t*>(base + pl.off_off);
  double* A = reinterpret_cast<double*>(base + pl.a_off);
  const long long dim = pl.dim, rows = pl.rows, ld = pl.dim;
  const long long a_stride = rows * dim;
  const double s = (double)h_scale;
  const double lam = 1.0 / ((double)C * s * s);
  const int c = n_classes;
  int rc;

  if (!pl.use_tc) {                 // the tensor-core Gram zeroes info together with its digit counts
    rc = lb_launch_zero_i32(h, d_info, n_cand, st);
    if (rc) return rc;
  }
  if (fs) {                         // streamed: only the exact tensor-core Gram with the fused right-hand side accumulates
    if (!(pl.primal && pl.use_tc && pl.fuse_rhs)) return LBCNN_ERR_INVALID_ARG;
    if (fs->stage == 1) {
      LbPhase ph(h, LBCNN_PHASE_GRAM, st);
      return lb_launch_gram_tc(h, base + pl.tc_off, d_H, n, F, n_cand, lam, A, a_stride, ld, true, d_labels, c, d_info, st,
                               fs->first_chunk == 0, fs->last_chunk != 0);
    }
  }

  if (fs && fs->stage == 2) {
    // the Gram and the right-hand side are complete in A
  } else if (pl.primal) {
    // F1: A = U^T U + lam I (lower tiles), operands read with k = sample (slow) and i = feature (contiguous)
    {
    LbPhase ph(h, LBCNN_PHASE_GRAM, st);
    if (pl.use_tc) {
      rc = lb_launch_gram_tc(h, base + pl.tc_off, d_H, n, F, n_cand, lam, A, a_stride, ld, true, d_labels, c, d_info, st);
      if (rc) return rc;
    } else {
    GemmP g{};
    g.A = d_H; g.sAr = 1; g.sAk = F; g.bA = n * F;
    g.B = d_H; g.sBr = 1; g.sBk = F; g.bB = n * F;
    g.C = A; g.ldc = ld; g.bC = a_stride;
    g.M = (int)F; g.N = (int)F; g.K = (int)n; g.alpha = 1.0; g.accumulate = 0; g.lower = 1; g.diag = lam;
    rc = launch_gemm<float, float, double, false, false>(h, g, n_cand, st);
    if (rc) return rc;
    }
    }
    // F2: appended rows = (U^T T)^T -- already written by the tensor-core Gram of [U | T]; otherwise label-segmented sums
    if (!pl.fuse_rhs) {
    LbPhase ph2(h, LBCNN_PHASE_RHS, st);
    label_perm_kernel<<<1, 1024, (c + 1) * sizeof(int), st>>>(d_labels, (int)n, c, perm, off);
    h->launches += 1;
    dim3 gr((unsigned)((F + 127) / 128), (unsigned)c, (unsigned)n_cand);
    rhs_primal_kernel<<<gr, 128, 0, st>>>(d_H, n, F, perm, off, A, a_stride, dim);
    h->launches += 1;
    }
  } else {
    {
    LbPhase ph(h, LBCNN_PHASE_GRAM, st);
    if (pl.use_tc) {
      rc = lb_launch_gram_tc(h, base + pl.tc_off, d_H, n, F, n_cand, lam, A, a_stride, ld, false, nullptr, 0, d_info, st, false, true,
                             n + pl.n_extra, c);
      if (rc) return rc;
    } else {
    GemmP g{};
    g.A = d_H; g.sAr = F; g.sAk = 1; g.bA = n * F;
    g.B = d_H; g.sBr = F; g.sBk = 1; g.bB = n * F;
    g.C = A; g.ldc = ld; g.bC = a_stride;
    g.M = (int)n; g.N = (int)n; g.K = (int)F; g.alpha = 1.0; g.accumulate = 0; g.lower = 1; g.diag = lam;
    rc = launch_gemm<float, float, double, true, true>(h, g, n_cand, st);
    if (rc) return rc;
    }
    }
    LbPhase ph2(h, LBCNN_PHASE_RHS, st);
    dim3 gr((unsigned)((n * c + 255) / 256), 1, (unsigned)n_cand);
    rhs_dual_kernel<<<gr, 256, 0, st>>>(d_labels, n, c, A, a_stride);
    h->launches += 1;
  }
  LB_CUDA_OK(cudaGetLastError());

  LbPhase ph3(h, LBCNN_PHASE_SOLVE, st);
  double* Linv = reinterpret_cast<double*>(base + pl.linv_off);
  const long long nblk = (dim + NB - 1) / NB;
  const long long linv_stride = nblk * NB * NB;

  // F3: right-looking blocked Cholesky over dim + c rows with two block sizes.  Inside a panel of NBO columns the
  // 64-column steps (factor the diagonal block and invert it; panel rows X = A21 L11^-T as a product; update the
  // REST OF THE PANEL only) touch a narrow strip; the wide trailing matrix is updated once per panel with K = NBO,
  // which cuts its read-modify-write traffic by NBO / NB.
  // With the tensor-core trailing update (chol_tc.cu) the wide update costs ~1/10 of its fp64 time, so the panel is made
  // wider (its read-modify-write traffic on the trailing matrix falls with 1/NBO).
  const bool tc_solve = pl.stc_kmax > 0 && (h->solver == LBCNN_SOLVER_MIXED || (h->solver == LBCNN_SOLVER_AUTO && pl.allow_tc && dim >= LB_STC_AUTO_DIM));
  const int NBO = tc_solve ? h->panel : 256;
  const int NBM = (tc_solve && h->mid_panel >= NB && h->mid_panel < NBO) ? h->mid_panel : NBO;      // mid level (fp64 steps inside)
  // columns of the common-mode deflation (fp64); never wider than one 64-column step or the system
  const int dfl = (tc_solve && h->deflate > 0) ? (int)((h->deflate < NB ? h->deflate : NB) < dim ? (h->deflate < NB ? h->deflate : NB) : dim) : 0;
  CholTcCtx tcx;
  if (tc_solve) {
    rc = lb_chol_tc_begin(h, base + pl.stc_off, rows, dim, n_cand, pl.stc_kmax, A, a_stride, ld, lb_ws_counter(h, 1), &tcx);
    if (rc) return rc;
  }
  const size_t potrf_smem = 2 * NB * (NB + 1) * sizeof(double);
  LB_CUDA_OK(cudaFuncSetAttribute(potrf_diag_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)potrf_smem));
  for (long long J0 = 0; J0 < dim; J0 += NBO) {
    const long long J1 = (J0 + NBO < dim) ? J0 + NBO : dim;
    for (long long j0 = J0; j0 < J1; j0 += NB) {
      const int nbj = (int)((dim - j0 < NB) ? dim - j0 : NB);
      double* Lj = Linv + (j0 / NB) * NB * NB;
      potrf_diag_kernel<<<n_cand, 256, potrf_smem, st>>>(A, a_stride, ld, (int)j0, nbj, d_info, Lj, linv_stride);
      h->launches += 1;
      const long long j1 = j0 + nbj;
      const long long M0 = J0 + (j0 - J0) / NBM * NBM, M1 = (M0 + NBM < J1) ? M0 + NBM : J1;     // the mid block of this step
      if (rows - j1 > 0) {
        GemmP g{};                                                     // X = A21 * Linv^T, in place (one column tile)
        g.A = A + j1 * ld + j0; g.sAr = ld; g.sAk = 1; g.bA = a_stride;
        g.B = Lj; g.sBr = NB; g.sBk = 1; g.bB = linv_stride;
        g.C = A + j1 * ld + j0; g.ldc = ld; g.bC = a_stride;
        g.M = (int)(rows - j1); g.N = nbj; g.K = nbj; g.alpha = 1.0; g.accumulate = 0; g.lower = 0; g.diag = 0.0;
        rc = launch_gemm<double, double, double, true, true>(h, g, n_cand, st);
        if (rc) return rc;
        // The very first columns carry the features' common mode (all features are positive: L's first column is 10-100x
        // larger than the rest of its row).  Inside a row-scaled int8 slice it would cost the other columns that many
        // bits, so the update of everything beyond the first mid block by the first `dfl` columns stays on the fp64 path
        // (a K = dfl product) and the tensor-core updates of block 0 / panel 0 start at column dfl.
        if (dfl > 0 && j0 == 0 && dim - M1 > 0) {
          GemmP u{};
          u.A = A + M1 * ld; u.sAr = ld; u.sAk = 1; u.bA = a_stride;
          u.B = A + M1 * ld; u.sBr = ld; u.sBk = 1; u.bB = a_stride;
          u.C = A + M1 * ld + M1; u.ldc = ld; u.bC = a_stride;
          u.M = (int)(rows - M1); u.N = (int)(dim - M1); u.K = dfl; u.alpha = -1.0; u.accumulate = 1; u.lower = 1; u.diag = 0.0;
          rc = launch_gemm<double, double, double, true, true>(h, u, n_cand, st);
          if (rc) return rc;
        }
        if (M1 - j1 > 0) {                                      // rest of the mid block: columns j1 .. M1-1 (fp64)
          GemmP u{};
          u.A = A + j1 * ld + j0; u.sAr = ld; u.sAk = 1; u.bA = a_stride;
          u.B = A + j1 * ld + j0; u.sBr = ld; u.sBk = 1; u.bB = a_stride;
          u.C = A + j1 * ld + j1; u.ldc = ld; u.bC = a_stride;
          u.M = (int)(rows - j1); u.N = (int)(M1 - j1); u.K = nbj; u.alpha = -1.0; u.accumulate = 1; u.lower = 1; u.diag = 0.0;
          rc = launch_gemm<double, double, double, true, true>(h, u, n_cand, st);
          if (rc) return rc;
        }
        // a finished mid block updates the rest of its panel on the tensor pipe (K = NBM): the fp64 steps above then only
        // ever touch NBM-wide strips, and the wide trailing matrix is read and written once per NBO columns
        if (j1 == M1 && J1 - M1 > 0 && NBM < NBO) {
          const long long K0 = (M0 == 0) ? dfl : M0;
          rc = lb_chol_tc_update(h, tcx, (int)M1, (int)J1, (int)K0, (int)(M1 - K0), st);
          if (rc) return rc;
        }
      }
    }
    if (dim - J1 > 0 && tc_solve) {                                    // trailing matrix on the tensor pipe
      const long long K0 = (J0 == 0) ? dfl : J0;                       // columns 0 .. dfl-1 were applied in fp64
      rc = lb_chol_tc_update(h, tcx, (int)J1, (int)dim, (int)K0, (int)(J1 - K0), st);
      if (rc) return rc;
    } else if (dim - J1 > 0) {                                         // trailing matrix, K = the whole panel
      GemmP g{};
      g.A = A + J1 * ld + J0; g.sAr = ld; g.sAk = 1; g.bA = a_stride;
      g.B = A + J1 * ld + J0; g.sBr = ld; g.sBk = 1; g.bB = a_stride;
      g.C = A + J1 * ld + J1; g.ldc = ld; g.bC = a_stride;
      g.M = (int)(rows - J1); g.N = (int)(dim - J1); g.K = (int)(J1 - J0); g.alpha = -1.0; g.accumulate = 1; g.lower = 1;
      g.diag = 0.0;
      rc = launch_gemm<double, double, double, true, true>(h, g, n_cand, st);
      if (rc) return rc;
    }
  }
  if (ds && pl.n_extra > 0) {
    // kernel trick (dual branch): the appended rows now hold Y_T = (L^-1 T)^T (c rows) and Y_te = (L^-1 K_te^T)^T (n_extra
    // rows, K_te = H_te U^T the exact cross-Gram), so  logits = K_te A^-1 T = Y_te Y_T^T  -- no W, no pass over H_te
    ph3.stop();
    {
      LbPhase phs(h, LBCNN_PHASE_SCORE, st);
      double* lg = reinterpret_cast<double*>(base + pl.lg_off);
      GemmP g{};
      g.A = A + (dim + c) * ld; g.sAr = ld; g.sAk = 1; g.bA = a_stride;
      g.B = A + dim * ld; g.sBr = ld; g.sBk = 1; g.bB = a_stride;
      g.C = lg; g.ldc = c; g.bC = pl.n_extra * c;
      g.M = (int)pl.n_extra; g.N = c; g.K = (int)dim; g.alpha = 1.0; g.accumulate = 0; g.lower = 0; g.diag = 0.0;
      rc = launch_gemm<double, double, double, true, true>(h, g, n_cand, st);
      if (rc) return rc;
      LB_CUDA_OK(cudaMemsetAsync(ds->correct, 0, (size_t)n_cand * 4, st));
      dim3 ga((unsigned)((pl.n_extra + 255) / 256), (unsigned)n_cand);
      dual_argmax_kernel<<<ga, 256, 0, st>>>(lg, pl.n_extra, c, ds->te_labels, ds->correct);
      h->launches += 1;
    }
  }
  LbPhase ph4(h, LBCNN_PHASE_SOLVE, st, ds && pl.n_extra > 0);      // a second bracket only when the scoring above split the phase
  // backward sweep on the appended rows: X^T L = Y^T, block columns from the last to the first;
  // the diagonal step is X_j = Y_j L_jj^-1 (a product with the stored inverse)
  for (long long jb = nblk - 1; jb >= 0; --jb) {
    const long long j0 = jb * NB;
    const int nbj = (int)((dim - j0 < NB) ? dim - j0 : NB);
    {
      GemmP g{};
      g.A = A + dim * ld + j0; g.sAr = ld; g.sAk = 1; g.bA = a_stride;
      g.B = Linv + jb * NB * NB; g.sBr = 1; g.sBk = NB; g.bB = linv_stride;   // B(j, k) = Linv[k][j]
      g.C = A + dim * ld + j0; g.ldc = ld; g.bC = a_stride;
      g.M = c; g.N = nbj; g.K = nbj; g.alpha = 1.0; g.accumulate = 0; g.lower = 0; g.diag = 0.0;
      rc = launch_gemm<double, double, double, true, false>(h, g, n_cand, st);
      if (rc) return rc;
    }
    if (j0 > 0) {
      GemmP g{};
      g.A = A + dim * ld + j0; g.sAr = ld; g.sAk = 1; g.bA = a_stride;      // X^T[:, block]  (c x nbj)
      g.B = A + j0 * ld; g.sBr = 1; g.sBk = ld; g.bB = a_stride;            // L[block, 0:j0] as (j, k)
      g.C = A + dim * ld; g.ldc = ld; g.bC = a_stride;
      g.M = c; g.N = (int)j0; g.K = nbj; g.alpha = -1.0; g.accumulate = 1; g.lower = 0; g.diag = 0.0;
      rc = launch_gemm<double, double, double, true, false>(h, g, n_cand, st);
      if (rc) return rc;
    }
  }
  LB_CUDA_OK(cudaGetLastError());

  if (pl.primal) {
    dim3 gw((unsigned)((dim * c + 255) / 256), 1, (unsigned)n_cand);
    w_from_xt_kernel<<<gw, 256, 0, st>>>(A, a_stride, dim, c, 1.0 / s, d_W);
    h->launches += 1;
  } else if (!(ds && pl.n_extra > 0)) {
    // W[f][cls] = (1/s) sum_n U[n][f] Z^T[cls][n]
    GemmP g{};
    g.A = d_H; g.sAr = 1; g.sAk = F; g.bA = n * F;
    g.B = A + dim * ld; g.sBr = ld; g.sBk = 1; g.bB = a_stride;
    g.C = d_W; g.ldc = c; g.bC = F * c;
    g.M = (int)F; g.N = c; g.K = (int)n; g.alpha = 1.0 / s; g.accumulate = 0; g.lower = 0; g.diag = 0.0;
    rc = launch_gemm<float, double, float, false, true>(h, g, n_cand, st);
    if (rc) return rc;
  }
  LB_CUDA_OK(cudaGetLastError());
  return LBCNN_OK;
}

