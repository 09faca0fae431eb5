// score.cu -- K4: fused logits + argmax + correct-count ("applied the feature vector directly
// to the Adaline output layer"; accuracy PAPER.md:23), and the search driver's final reduction.
//
// The output layer is skinny (c = 10..100 classes), so this is not a tile GEMM: one CTA owns 64 test rows of one
// candidate, stages 64 x 64 tiles of H (coalesced float4 loads) and the matching 64 x (16 NCH) slab of W in
// shared memory (widened to fp64 once per tile), and every thread keeps 8 NCH fp64 logits of ONE row in registers
// (two threads per row; up to 64 classes per pass).  The
// products are fp32 x fp32 widened to fp64 (exact), the sums fp64 -- the same arithmetic as the oracle's fp64
// logits up to summation order; the argmax (first index on ties) and the correct count never leave the CTA.
#include "internal.h"

namespace {

constexpr int SC_ROWS = 64, SC_KT = 64, SC_THREADS = 128, SC_LDH = SC_KT + 1;

template <int NCH>
__global__ void __launch_bounds__(SC_THREADS) score_kernel(const float* __restrict__ U, long long n, long long F, double hs,
                                                           const float* __restrict__ W, int c, const int32_t* __restrict__ y,
                                                           int32_t* __restrict__ pred, int32_t* __restrict__ correct) {
  constexpr int CW = 16 * NCH;                       // classes per pass
  extern __shared__ __align__(16) double sc_smem[];     // widened once per tile: F2F in the inner loop would bound it
  double* Hs = sc_smem;                                 // [SC_ROWS][SC_LDH]
  double* Ws = sc_smem + SC_ROWS * SC_LDH;              // [SC_KT][CW], 16-byte aligned (SC_ROWS * SC_LDH is even)
  __shared__ int s_ok;
  const long long z = blockIdx.y;
  const long long i0 = (long long)blockIdx.x * SC_ROWS;
  const float* Uz = U + z * n * F;
  const float* Wz = W + z * F * c;
  const int t = threadIdx.x, r = t >> 1, h = t & 1;
  if (t == 0) s_ok = 0;
  double best = 0.0;
  int bidx = -1;
  const bool vec = ((F & 3) == 0) && ((reinterpret_cast<uintptr_t>(Uz) & 15) == 0);
  for (int cc0 = 0; cc0 < c; cc0 += CW) {
    double acc[NCH][8];
#pragma unroll
    for (int q = 0; q < NCH; ++q)
#pragma unroll
      for (int e = 0; e < 8; ++e) acc[q][e] = 0.0;
    for (long long k0 = 0; k0 < F; k0 += SC_KT) {
      __syncthreads();                               // previous tile fully consumed
      if (vec) {
#pragma unroll
        for (int q = 0; q < SC_ROWS * SC_KT / 4 / SC_THREADS; ++q) {
          const int idx = t + SC_THREADS * q, row = idx >> 4, f4 = (idx & 15) * 4;
          float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
          if (i0 + row < n && k0 + f4 < F) v = __ldcs(reinterpret_cast<const float4*>(Uz + (i0 + row) * F + k0 + f4));
          double* d = Hs + row * SC_LDH + f4;
          d[0] = (double)v.x; d[1] = (double)v.y; d[2] = (double)v.z; d[3] = (double)v.w;
        }
      } else {
        for (int idx = t; idx < SC_ROWS * SC_KT; idx += SC_THREADS) {
          const int row = idx >> 6, f = idx & 63;
          Hs[row * SC_LDH + f] = (i0 + row < n && k0 + f < F) ? (double)Uz[(i0 + row) * F + k0 + f] : 0.0;
        }
      }
      for (int idx = t; idx < SC_KT * CW; idx += SC_THREADS) {
        const int kf = idx / CW, cc = idx - kf * CW;
        Ws[idx] = (k0 + kf < F && cc0 + cc < c) ? (double)Wz[(k0 + kf) * c + cc0 + cc] : 0.0;
      }
      __syncthreads();
#pragma unroll 4
      for (int kf = 0; kf < SC_KT; ++kf) {
        const double hv = Hs[r * SC_LDH + kf];
#pragma unroll
        for (int q = 0; q < NCH; ++q) {
          const double2* wp = reinterpret_cast<const double2*>(Ws + kf * CW + q * 16 + h * 8);
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const double2 w = wp[e];
            acc[q][2 * e] = fma(hv, w.x, acc[q][2 * e]);
            acc[q][2 * e + 1] = fma(hv, w.y, acc[q][2 * e + 1]);
          }
        }
      }
    }
    // classes of this thread in increasing index order within a chunk; strict '>' keeps the lowest index on ties
#pragma unroll
    for (int q = 0; q < NCH; ++q)
#pragma unroll
      for (int e = 0; e < 8; ++e) {
        const int j = cc0 + q * 16 + h * 8 + e;
        const double l = hs * acc[q][e];
        if (j < c && (bidx < 0 || l > best || (l == best && j < bidx))) { best = l; bidx = j; }
      }
  }
  {  // the two threads of a row: larger logit wins, the lower class index on equality (R12)
    const double ov = __shfl_xor_sync(0xffffffffu, best, 1);
    const int oi = __shfl_xor_sync(0xffffffffu, bidx, 1);
    if (oi >= 0 && (bidx < 0 || ov > best || (ov == best && oi < bidx))) { best = ov; bidx = oi; }
  }
  int ok = 0;
  if (h == 0 && i0 + r < n) {
    if (pred) pred[z * n + i0 + r] = bidx;
    if (y && y[i0 + r] == bidx) ok = 1;
  }
  __syncthreads();
  ok = __reduce_add_sync(0xffffffffu, ok);
  if ((t & 31) == 0 && ok) atomicAdd(&s_ok, ok);
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

}  // namespace

int lb_launch_score(lbcnn_handle_s* h, const float* d_H, int64_t n, int64_t F, float h_scale, const float* d_W,
                    int n_classes, const int32_t* d_labels, int n_cand, int32_t* d_pred, int32_t* d_correct,
                    cudaStream_t st) {
  LbPhase ph(h, LBCNN_PHASE_SCORE, st);
  if (d_correct) {
    int rc = lb_launch_zero_i32(h, d_correct, n_cand, st);
    if (rc) return rc;
  }
  dim3 grid((unsigned)((n + SC_ROWS - 1) / SC_ROWS), (unsigned)n_cand);
  const int nch = (n_classes + 15) / 16;             // 16-class chunks; a pass keeps up to four of them in registers
  const double hs = (double)h_scale;
#define LB_SCORE(NCH)                                                                                                     \
  do {                                                                                                                    \
    const size_t sm = sizeof(double) * (SC_ROWS * SC_LDH + SC_KT * 16 * NCH);                                         \
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
