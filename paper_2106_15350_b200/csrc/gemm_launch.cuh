// gemm_launch.cuh -- the batched fp64-accumulating GEMM launcher on top of the DMMA tile engine (gemm64.cuh), shared by the
// fit (fit.cu) and the output-layer refinement (refine.cu).  Header-only templates; include inside the library only.
#pragma once
#include "internal.h"
#include "gemm64.cuh"

namespace {

// generic batched GEMM, fp64 accumulate:  C[i][j] (+)= alpha * sum_k A(i,k) B(j,k) (+ diag on i == j)
struct GemmP {
  const void* A; long long sAr, sAk, bA;
  const void* B; long long sBr, sBk, bB;
  void* C; long long ldc, bC;
  int M, N, K;
  double alpha; int accumulate; int lower; double diag;
};

template <typename TA, typename TB, typename TC, bool AK, bool BK>
__global__ void __launch_bounds__(g64::NT) gemm_kernel(const GemmP p) {
  const int ti = blockIdx.y, tj = blockIdx.x;
  if (p.lower && tj > ti) return;
  __shared__ g64::Smem sm;
  const long long z = blockIdx.z;
  const TA* A = reinterpret_cast<const TA*>(p.A) + z * p.bA;
  const TB* B = reinterpret_cast<const TB*>(p.B) + z * p.bB;
  TC* C = reinterpret_cast<TC*>(p.C) + z * p.bC;
  double acc[2][4][2];
  g64::tile_mma<TA, TB, AK, BK>(sm, A, p.sAr, p.sAk, ti * 64, p.M, B, p.sBr, p.sBk, tj * 64, p.N, p.K, acc);
#pragma unroll
  for (int m = 0; m < 2; ++m) {
    const int i = ti * 64 + g64::frag_row(m);
    if (i >= p.M) continue;
#pragma unroll
    for (int nb = 0; nb < 4; ++nb)
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int j = tj * 64 + g64::frag_col(nb, e);
        if (j >= p.N) continue;
        double v = p.alpha * acc[m][nb][e];
        if (i == j) v += p.diag;
        TC* c = C + (long long)i * p.ldc + j;
        if (p.accumulate) v += (double)*c;
        *c = (TC)v;
      }
  }
}

template <typename TA, typename TB, typename TC, bool AK, bool BK>
int launch_gemm(lbcnn_handle_s* h, const GemmP& p, int batch, cudaStream_t st) {
  if (p.M <= 0 || p.N <= 0 || batch <= 0) return LBCNN_OK;
  dim3 grid((p.N + 63) / 64, (p.M + 63) / 64, batch);
  gemm_kernel<TA, TB, TC, AK, BK><<<grid, g64::NT, 0, st>>>(p);
  h->launches += 1;
  LB_CUDA_OK(cudaGetLastError());
  return LBCNN_OK;
}


}  // namespace
