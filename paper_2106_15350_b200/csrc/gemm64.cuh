// gemm64.cuh -- 64x64x16 tile engine with fp64 accumulation (SIMT DFMA), operands fp32 or fp64.
// acc[qi][qj] = sum_k A(i,k) * B(j,k) for i = i0 + ty + 16*qi, j = j0 + tx + 16*qj.
// Operand element (r,k) lives at base[r*s_r + k*s_k]; KCONTIG says which of the two strides is 1, which
// only selects the thread->element mapping of the global loads (coalescing), not the result.
// Products of two fp32 numbers are exact in fp64, so for integer-valued H (abs < 2^24) the Gram sums
// are exact as long as they stay below 2^53.
#pragma once
#include <cuda_runtime.h>

namespace g64 {

constexpr int TM = 64, TN = 64, TK = 16, LD = 66, NT = 256;

struct Smem {
  double a[TK][LD];
  double b[TK][LD];
};

// load one 64 x 16 operand tile into registers (4 elements per thread), zero outside [0,R) x [0,K)
template <typename T, bool KCONTIG>
__device__ __forceinline__ void load_tile(const T* __restrict__ base, long long s_r, long long s_k, int r0, int R,
                                          int k0, int K, double v[4]) {
  const int t = threadIdx.x;
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const int e = t + NT * q;
    int r, k;
    if (KCONTIG) { r = e >> 4; k = e & 15; } else { k = e >> 6; r = e & 63; }
    const int gr = r0 + r, gk = k0 + k;
    v[q] = (gr < R && gk < K) ? (double)base[(long long)gr * s_r + (long long)gk * s_k] : 0.0;
  }
}

template <bool KCONTIG>
__device__ __forceinline__ void store_tile(double (*s)[LD], const double v[4]) {
  const int t = threadIdx.x;
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const int e = t + NT * q;
    int r, k;
    if (KCONTIG) { r = e >> 4; k = e & 15; } else { k = e >> 6; r = e & 63; }
    s[k][r] = v[q];
  }
}

template <typename TA, typename TB, bool AK, bool BK>
__device__ __forceinline__ void tile_mma(Smem& sm, const TA* __restrict__ A, long long sAr, long long sAk, int i0,
                                         int M, const TB* __restrict__ B, long long sBr, long long sBk, int j0, int N,
                                         int K, double acc[4][4]) {
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) acc[a][b] = 0.0;
  double va[4], vb[4];
  load_tile<TA, AK>(A, sAr, sAk, i0, M, 0, K, va);
  load_tile<TB, BK>(B, sBr, sBk, j0, N, 0, K, vb);
  for (int k0 = 0; k0 < K; k0 += TK) {
    __syncthreads();                       // previous tile fully consumed
    store_tile<AK>(sm.a, va);
    store_tile<BK>(sm.b, vb);
    __syncthreads();
    if (k0 + TK < K) {                     // prefetch the next tile while computing this one
      load_tile<TA, AK>(A, sAr, sAk, i0, M, k0 + TK, K, va);
      load_tile<TB, BK>(B, sBr, sBk, j0, N, k0 + TK, K, vb);
    }
#pragma unroll
    for (int kk = 0; kk < TK; ++kk) {
      double ra[4], rb[4];
#pragma unroll
      for (int q = 0; q < 4; ++q) { ra[q] = sm.a[kk][ty + 16 * q]; rb[q] = sm.b[kk][tx + 16 * q]; }
#pragma unroll
      for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) acc[a][b] = fma(ra[a], rb[b], acc[a][b]);
    }
  }
}

}  // namespace g64
