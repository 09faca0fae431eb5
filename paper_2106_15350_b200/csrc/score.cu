// score.cu -- K4: fused logits + argmax + correct-count ("applied the feature vector directly
// to the Adaline output layer"; accuracy PAPER.md:23), and the search driver's final reduction.
//
// The output layer is skinny (c = 10..100 classes) and the logits are wanted in fp64 (the oracle's arithmetic; with
// 120-sample test sets a single flipped near-tie already breaks label parity), so this runs on the fp64 tensor
// path: mma.sync m8n8k4 (DMMA, 64 fp64 FMA/clk/SM on B200 -- the same peak as DFMA but one instruction per 256 FMAs
// and operands reused from registers, where the plain DFMA loop was bound by shared-memory bandwidth).
// One CTA owns 128 test rows of one candidate; a warp owns 32 rows x (16 NCH) classes of accumulators.  H tiles
// (128 x 32, coalesced float4 loads) and the matching W slab are widened to fp64 once when staged into shared
// memory (products of two fp32 numbers are exact in fp64); the argmax (first index on ties) and the correct count
// never leave the CTA.
#include "internal.h"

namespace {

constexpr int SC_ROWS = 128, SC_KT = 32, SC_THREADS = 128;
constexpr int SC_LDH = SC_KT + 4;        // row pitch of the H tile in doubles: = 4 (mod 16) -> conflict-free A fragments

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

template <int NCH>
__global__ void __launch_bounds__(SC_THREADS) score_kernel(const float* __restrict__ U, long long n, long long F, double hs,
                                                           const float* __restrict__ W, int c, const int32_t* __restrict__ y,
                                                           int32_t* __restrict__ pred, int32_t* __restrict__ correct) {
  constexpr int CW = 16 * NCH;             // classes per pass
  constexpr int LDW = CW + 8;              // pitch of the W slab: = 8 (mod 16) -> conflict-free B fragments
  extern __shared__ __align__(16) double sc_smem[];
  double* Hs = sc_smem;                    // [SC_ROWS][SC_LDH]
  double* Ws = sc_smem + SC_ROWS * SC_LDH; // [SC_KT][LDW]
  __shared__ int s_ok;
  const long long z = blockIdx.y;
  const long long i0 = (long long)blockIdx.x * SC_ROWS;
  const float* Uz = U + z * n * F;
  const float* Wz = W + z * F * c;
  const int t = threadIdx.x, warp = t >> 5, lane = t & 31;
  const int g = lane >> 2, q4 = lane & 3;  // fragment coordinates: row / column group and k index
  if (t == 0) s_ok = 0;
  double best[4];
  int bidx[4];
#pragma unroll
  for (int m = 0; m < 4; ++m) { best[m] = 0.0; bidx[m] = -1; }
  const bool vec = ((F & 3) == 0) && ((reinterpret_cast<uintptr_t>(Uz) & 15) == 0);
  for (int cc0 = 0; cc0 < c; cc0 += CW) {
    double acc[4][2 * NCH][2];             // [row block of 8][class block of 8][2 columns]
#pragma unroll
    for (int m = 0; m < 4; ++m)
#pragma unroll
      for (int nb = 0; nb < 2 * NCH; ++nb) { acc[m][nb][0] = 0.0; acc[m][nb][1] = 0.0; }
    for (long long k0 = 0; k0 < F; k0 += SC_KT) {
      __syncthreads();                     // previous tile fully consumed
      if (vec) {
#pragma unroll
        for (int q = 0; q < SC_ROWS * SC_KT / 4 / SC_THREADS; ++q) {
          const int idx = t + SC_THREADS * q, row = idx >> 3, f4 = (idx & 7) * 4;
          float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
          if (i0 + row < n && k0 + f4 < F) v = __ldcs(reinterpret_cast<const float4*>(Uz + (i0 + row) * F + k0 + f4));
          double2* d = reinterpret_cast<double2*>(Hs + row * SC_LDH + f4);
          d[0] = make_double2((double)v.x, (double)v.y);
          d[1] = make_double2((double)v.z, (double)v.w);
        }
      } else {
        for (int idx = t; idx < SC_ROWS * SC_KT; idx += SC_THREADS) {
          const int row = idx >> 5, f = idx & 31;
          Hs[row * SC_LDH + f] = (i0 + row < n && k0 + f < F) ? (double)Uz[(i0 + row) * F + k0 + f] : 0.0;
        }
      }
      for (int idx = t; idx < SC_KT * CW; idx += SC_THREADS) {
        const int kf = idx / CW, cc = idx - kf * CW;
        Ws[kf * LDW + cc] = (k0 + kf < F && cc0 + cc < c) ? (double)Wz[(k0 + kf) * c + cc0 + cc] : 0.0;
      }
      __syncthreads();
      const double* ha = Hs + (warp * 32 + g) * SC_LDH + q4;
      const double* wb = Ws + q4 * LDW + g;
#pragma unroll
      for (int k4 = 0; k4 < SC_KT; k4 += 4) {
        double a[4], b[2 * NCH];
#pragma unroll
        for (int m = 0; m < 4; ++m) a[m] = ha[m * 8 * SC_LDH + k4];
#pragma unroll
        for (int nb = 0; nb < 2 * NCH; ++nb) b[nb] = wb[k4 * LDW + nb * 8];
#pragma unroll
        for (int m = 0; m < 4; ++m)
#pragma unroll
          for (int nb = 0; nb < 2 * NCH; ++nb) dmma884(acc[m][nb][0], acc[m][nb][1], a[m], b[nb]);
      }
    }
    // this lane's classes of row (warp*32 + 8m + g): 8nb + 2 q4 + {0,1}, visited in increasing index order
#pragma unroll
    for (int m = 0; m < 4; ++m)
#pragma unroll
      for (int nb = 0; nb < 2 * NCH; ++nb)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int j = cc0 + nb * 8 + 2 * q4 + e;
          const double l = hs * acc[m][nb][e];
          if (j < c && (bidx[m] < 0 || l > best[m] || (l == best[m] && j < bidx[m]))) { best[m] = l; bidx[m] = j; }
        }
  }
  // the four lanes of a row: larger logit wins, the lower class index on equality (R12)
  int ok = 0;
#pragma unroll
  for (int m = 0; m < 4; ++m) {
#pragma unroll
    for (int d = 1; d <= 2; d <<= 1) {
      const double ov = __shfl_xor_sync(0xffffffffu, best[m], d);
      const int oi = __shfl_xor_sync(0xffffffffu, bidx[m], d);
      if (oi >= 0 && (bidx[m] < 0 || ov > best[m] || (ov == best[m] && oi < bidx[m]))) { best[m] = ov; bidx[m] = oi; }
    }
    const long long i = i0 + warp * 32 + m * 8 + g;
    if (q4 == 0 && i < n) {
      if (pred) pred[z * n + i] = bidx[m];
      if (y && y[i] == bidx[m]) ok += 1;
    }
  }
  __syncthreads();
  ok = __reduce_add_sync(0xffffffffu, ok);
  if (lane == 0 && ok) atomicAdd(&s_ok, ok);
  __syncthreads();
  if (t == 0 && correct && s_ok) atomicAdd(&correct[z], s_ok);
}

__global__ void zero_i32_kernel(int32_t* p, long long n) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t < n) p[t] = 0;
}

// acc[k] = correct/n_test or -1; best = first maximum, worst = first minimum among successful fits;
// W_best = W of the best candidate.
__global__ void finish_kernel(const int32_t* __restrict__ correct, const int32_t* __restrict__ info, long long n_test,
                              int n_cand, float* __restrict__ acc, int32_t* __restrict__ best,
                              const float* __restrict__ W_all, long long w_elems, float* __restrict__ W_best) {
  __shared__ int s_best;
  for (int k = threadIdx.x; k < n_cand; k += blockDim.x)
    acc[k] = info[k] ? -1.0f : (float)((double)correct[k] / (double)n_test);
  __syncthreads();
  if (threadIdx.x == 0) {
    int b = -1, w = -1;
    for (int k = 0; k < n_cand; ++k) {
      if (info[k]) continue;
      if (b < 0 || correct[k] > correct[b]) b = k;
      if (w < 0 || correct[k] < correct[w]) w = k;
    }
    if (b < 0) { b = 0; w = 0; }
    best[0] = b; best[1] = w;
    s_best = b;
  }
  __syncthreads();
  if (W_best && W_all) {
    const float* src = W_all + (long long)s_best * w_elems;
    for (long long t = threadIdx.x; t < w_elems; t += blockDim.x) W_best[t] = src[t];
  }
}

// kernel set (and bias) of candidate best[0] copied to a slot of its own: a chunked dual-branch search re-fits its best
// candidate after the last chunk, and the index exists on the device only
__global__ void gather_best_kernel(const int32_t* __restrict__ best, const int8_t* __restrict__ ker, long long nw,
                                   const int32_t* __restrict__ bias, long long nb, int8_t* __restrict__ ker_out,
                                   int32_t* __restrict__ bias_out) {
  const long long b = best[0];
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t < nw) ker_out[t] = ker[b * nw + t];
  if (bias && t < nb) bias_out[t] = bias[b * nb + t];
}

}  // namespace

int lb_launch_gather_best(lbcnn_handle_s* h, const int32_t* d_best, const int8_t* d_kernels, int64_t n_weights,
                          const int32_t* d_bias, int64_t n_bias, int8_t* ker_out, int32_t* bias_out, cudaStream_t st) {
  const int64_t m = n_weights > n_bias ? n_weights : n_bias;
  gather_best_kernel<<<(unsigned)((m + 255) / 256), 256, 0, st>>>(d_best, d_kernels, n_weights, d_bias, n_bias, ker_out, bias_out);
  h->launches += 1;
  LB_CUDA_OK(cudaGetLastError());
  return LBCNN_OK;
}

int lb_launch_score(lbcnn_handle_s* h, const float* d_H, int64_t n, int64_t F, float h_scale, const float* d_W,
                    int n_classes, const int32_t* d_labels, int n_cand, int32_t* d_pred, int32_t* d_correct,
                    cudaStream_t st, bool keep_correct) {
  LbPhase ph(h, LBCNN_PHASE_SCORE, st);
  if (d_correct && !keep_correct) {
    int rc = lb_launch_zero_i32(h, d_correct, n_cand, st);
    if (rc) return rc;
  }
  dim3 grid((unsigned)((n + SC_ROWS - 1) / SC_ROWS), (unsigned)n_cand);
  const int nch = (n_classes + 15) / 16;             // 16-class chunks; a pass keeps up to four of them in registers
  const double hs = (double)h_scale;
#define LB_SCORE(NCH)                                                                                                     \
  do {                                                                                                                    \
    const size_t sm = sizeof(double) * (SC_ROWS * SC_LDH + SC_KT * (16 * NCH + 8));                                         \
    LB_CUDA_OK(cudaFuncSetAttribute(score_kernel<NCH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));            \
    score_kernel<NCH><<<grid, SC_THREADS, sm, st>>>(d_H, n, F, hs, d_W, n_classes, d_labels, d_pred, d_correct);         \
  } while (0)
  if (nch == 1) LB_SCORE(1);
  else if (nch == 2) LB_SCORE(2);
  else if (nch == 3) LB_SCORE(3);
  else LB_SCORE(4);
#undef LB_SCORE
  h->launches += 1;
  LB_CUDA_OK(cudaGetLastError());
  return LBCNN_OK;
}

int lb_launch_zero_i32(lbcnn_handle_s* h, int32_t* p, int64_t n, cudaStream_t st) {
  zero_i32_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(p, n);
  h->launches += 1;
  LB_CUDA_OK(cudaGetLastError());
  return LBCNN_OK;
}

int lb_launch_finish(lbcnn_handle_s* h, const int32_t* d_correct, const int32_t* d_info, int64_t n_test, int n_cand,
                     float* d_acc, int32_t* d_best, const float* d_W_all, int64_t w_elems, float* d_W_best,
                     cudaStream_t st) {
  LbPhase ph(h, LBCNN_PHASE_FINISH, st);
  finish_kernel<<<1, 1024, 0, st>>>(d_correct, d_info, n_test, n_cand, d_acc, d_best, d_W_all, w_elems, d_W_best);
  h->launches += 1;
  LB_CUDA_OK(cudaGetLastError());
  return LBCNN_OK;
}
