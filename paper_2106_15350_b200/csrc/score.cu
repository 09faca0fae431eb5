// score.cu -- K4: fused logits + argmax + correct-count ("applied the feature vector directly
// to the Adaline output layer"; accuracy PAPER.md:23), and the search driver's final reduction.
//
// One CTA owns 64 test rows of one candidate and walks the classes in chunks of 64 with the fp64 tile
// engine; the argmax never leaves registers (column-wise best per thread, then a 16-lane shuffle
// reduction that prefers the larger value and, on equality, the lower class index).
#include "internal.h"
#include "gemm64.cuh"

namespace {

__global__ void __launch_bounds__(g64::NT) score_kernel(const float* __restrict__ U, long long n, long long F,
                                                        double hs, const float* __restrict__ W, int c,
                                                        const int32_t* __restrict__ y, int32_t* __restrict__ pred,
                                                        int32_t* __restrict__ correct) {
  __shared__ g64::Smem sm;
  __shared__ int s_ok;
  const long long z = blockIdx.y;
  const int i0 = blockIdx.x * 64;
  const float* Uz = U + z * n * F;
  const float* Wz = W + z * F * c;
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  if (threadIdx.x == 0) s_ok = 0;
  double best[4];
  int bidx[4];
#pragma unroll
  for (int a = 0; a < 4; ++a) { best[a] = 0.0; bidx[a] = -1; }
  for (int j0 = 0; j0 < c; j0 += 64) {
    double acc[4][4];
    g64::tile_mma<float, float, true, false>(sm, Uz, F, 1, i0, (int)n, Wz, 1, c, j0, c, (int)F, acc);
#pragma unroll
    for (int a = 0; a < 4; ++a) {
      double v = 0.0; int idx = -1;
#pragma unroll
      for (int b = 0; b < 4; ++b) {
        const int j = j0 + tx + 16 * b;
        const double l = hs * acc[a][b];
        if (j < c && (idx < 0 || l > v)) { v = l; idx = j; }
      }
#pragma unroll
      for (int d = 8; d >= 1; d >>= 1) {
        const double ov = __shfl_xor_sync(0xffffffffu, v, d);
        const int oi = __shfl_xor_sync(0xffffffffu, idx, d);
        if (oi >= 0 && (idx < 0 || ov > v || (ov == v && oi < idx))) { v = ov; idx = oi; }
      }
      if (idx >= 0 && (bidx[a] < 0 || v > best[a])) { best[a] = v; bidx[a] = idx; }   // later chunks have larger indices
    }
  }
  int ok = 0;
  if (tx == 0) {
#pragma unroll
    for (int a = 0; a < 4; ++a) {
      const long long i = i0 + ty + 16 * a;
      if (i < n) {
        if (pred) pred[z * n + i] = bidx[a];
        if (y && y[i] == bidx[a]) ok += 1;
      }
    }
  }
  __syncthreads();
  if (ok) atomicAdd(&s_ok, ok);
  __syncthreads();
  if (threadIdx.x == 0 && correct && s_ok) atomicAdd(&correct[z], s_ok);
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
  dim3 grid((unsigned)((n + 63) / 64), (unsigned)n_cand);
  score_kernel<<<grid, g64::NT, 0, st>>>(d_H, n, F, (double)h_scale, d_W, n_classes, d_labels, d_pred, d_correct);
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
