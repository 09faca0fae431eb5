// gemm64.cuh -- 64x64x16 tile engine with fp64 accumulation on the fp64 tensor path (mma.sync m8n8k4, DMMA),
// operands fp32 or fp64.  Eight warps; warp w owns rows 16 (w & 3) .. +15 and columns 32 (w >> 2) .. +31 as
// 2 x 4 fragments:  acc[m][nb][e] = sum_k A(i,k) * B(j,k)  for  i = i0 + row(m),  j = j0 + col(nb, e)  (see
// frag_row / frag_col).  DMMA has the same peak as DFMA on B200 (64 FMA/clk/SM) but takes its operands from
// registers that are reused across fragments, so the loop is no longer bound by shared-memory bandwidth.
// Operand element (r,k) lives at base[r*s_r + k*s_k]; KCONTIG says which of the two strides is 1, which
// only selects the thread->element mapping of the global loads (coalescing), not the result.
// Products of two fp32 numbers are exact in fp64, so for integer-valued H (abs < 2^24) the Gram sums
// are exact as long as they stay below 2^53.
#pragma once
#include <cuda_runtime.h>

namespace g64 {

constexpr int TM = 64, TN = 64, TK = 16, LD = 73, NT = 256;   // odd pitch: the transposing tile stores and the fragment loads both stay (nearly) conflict-free

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

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
// tile coordinates of accumulator (m, nb, e) of the calling thread
__device__ __forceinline__ int frag_row(int m) { return ((threadIdx.x >> 5) & 3) * 16 + m * 8 + ((threadIdx.x & 31) >> 2); }
__device__ __forceinline__ int frag_col(int nb, int e) { return (threadIdx.x >> 7) * 32 + nb * 8 + 2 * (threadIdx.x & 3) + e; }

template <typename TA, typename TB, bool AK, bool BK>
__device__ __forceinline__ void tile_mma(Smem& sm, const TA* __restrict__ A, long long sAr, long long sAk, int i0,
                                         int M, const TB* __restrict__ B, long long sBr, long long sBk, int j0, int N,
                                         int K, double acc[2][4][2]) {
  const int warp = threadIdx.x >> 5, g = (threadIdx.x & 31) >> 2, q4 = threadIdx.x & 3;
  const int ra = (warp & 3) * 16 + g, cb = (warp >> 2) * 32 + g;
#pragma unroll
  for (int m = 0; m < 2; ++m)
#pragma unroll
    for (int nb = 0; nb < 4; ++nb) { acc[m][nb][0] = 0.0; acc[m][nb][1] = 0.0; }
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
    for (int k4 = 0; k4 < TK; k4 += 4) {
      double fa[2], fb[4];
#pragma unroll
      for (int m = 0; m < 2; ++m) fa[m] = sm.a[k4 + q4][ra + 8 * m];
#pragma unroll
      for (int nb = 0; nb < 4; ++nb) fb[nb] = sm.b[k4 + q4][cb + 8 * nb];
#pragma unroll
      for (int m = 0; m < 2; ++m)
#pragma unroll
        for (int nb = 0; nb < 4; ++nb) dmma884(acc[m][nb][0], acc[m][nb][1], fa[m], fb[nb]);
    }
  }
}

}  // namespace g64
