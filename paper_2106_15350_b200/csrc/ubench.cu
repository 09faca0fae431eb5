// ubench.cu -- microbenchmarks behind the kernel designs: what one tcgen05.mma kind::i8 costs as a
// function of N and of the operand layout, what a tcgen05.ld round trip costs, and the fp64 DMMA rate.  A stand-alone
// program (built and run by `python -m paper_2106_15350_b200.ubench`), not part of liblbcnn.so.  One CTA, clock64() around
// a chain of back-to-back instructions of one kind; operands are whatever shared memory holds (timing does not depend on
// the values), every MMA accumulates into the same TMEM columns.
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
#include "tc_common.cuh"

namespace {

constexpr int REPS = 512;

// layout: 0 = K-major no swizzle (8-row core matrices 128 B apart), 1 = same but the start shifted by one row (16 B),
//         4 = K-major 64-byte swizzle, 2 = K-major 128-byte swizzle
template <int NACC>
__global__ void __launch_bounds__(128, 1) mma_i8_kernel(int N, int layout, long long* out) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t bar;
  __shared__ uint32_t tmem_base_s;
  const int warp = tc::uniform_warp_id(), lane = threadIdx.x & 31;
  for (int i = threadIdx.x; i < 64 * 1024 / 4; i += blockDim.x) reinterpret_cast<uint32_t*>(smem)[i] = 0x01010101u * (i & 3);
  if (threadIdx.x == 0) { tc::mbar_init(tc::smem_u32(&bar), 1); tc::fence_barrier_init(); }
  if (warp == 0) tc::tmem_alloc(tc::smem_u32(&tmem_base_s), 512);
  tc::fence_proxy_async();
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t tmem = tmem_base_s;
  if (warp == 0) {
    const uint32_t a0 = tc::smem_u32(smem) + (layout == 1 ? 16u : 0u), b0 = tc::smem_u32(smem) + 32 * 1024 + (layout == 1 ? 16u : 0u);
    uint64_t da, db;
    if (layout == 0 || layout == 1) {          // no swizzle: K chunk (16 B) stride = rows * 16, 8-row group stride 128 B
      da = tc::smem_desc(a0, 128 * 16, 128, tc::LAYOUT_NONE);
      db = tc::smem_desc(b0, (uint32_t)N * 16, 128, tc::LAYOUT_NONE);
    } else if (layout == 4) {
      da = tc::smem_desc(a0, 16, 512, 4);
      db = tc::smem_desc(b0, 16, 512, 4);
    } else {
      da = tc::smem_desc(a0, 16, 1024, tc::LAYOUT_SW128);
      db = tc::smem_desc(b0, 16, 1024, tc::LAYOUT_SW128);
    }
    const uint32_t idesc = tc::idesc_i8(128, N, 1, 1, 0, 0);
    // warm-up chain, then the timed chain
    for (int pass = 0; pass < 2; ++pass) {
      const long long t0 = clock64();
      for (int r = 0; r < REPS; r += NACC) {
#pragma unroll
        for (int q = 0; q < NACC; ++q)
          if (tc::elect_one()) tc::mma_i8(tmem + (uint32_t)(q * N), da, db, idesc, 1u);
      }
      if (tc::elect_one()) tc::mma_commit(tc::smem_u32(&bar));
      __syncwarp();
      tc::mbar_wait(tc::smem_u32(&bar), pass & 1);
      const long long t1 = clock64();
      if (pass == 1 && lane == 0) out[0] = t1 - t0;
    }
  }
  tc::tc_fence_before();
  __syncthreads();
  if (warp == 0) { tc::tc_fence_after(); tc::tmem_dealloc(tmem, 512); }
}

// tcgen05.ld 32x32b.x16: `inflight` loads issued before each wait, by `nwarps` warps (each its own lane quarter)
__global__ void __launch_bounds__(512, 1) tmem_ld_kernel(int inflight, long long* out) {
  __shared__ uint32_t tmem_base_s;
  const int warp = tc::uniform_warp_id(), lane = threadIdx.x & 31;
  if (warp == 0) tc::tmem_alloc(tc::smem_u32(&tmem_base_s), 512);
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t taddr = tmem_base_s + ((uint32_t)((warp & 3) * 32) << 16);
  uint32_t sink = 0;
  __syncthreads();
  const long long t0 = clock64();
  for (int r = 0; r < REPS; r += inflight) {
    uint32_t v[4][16];
#pragma unroll
    for (int q = 0; q < 4; ++q)
      if (q < inflight) tc::tmem_ld16(taddr + ((r + q) & 31) * 16, v[q]);
    tc::tmem_ld_wait();
#pragma unroll
    for (int q = 0; q < 4; ++q)
      if (q < inflight) sink ^= v[q][0] ^ v[q][15];
  }
  const long long t1 = clock64();
  __syncthreads();
  if (threadIdx.x == 0) { out[0] = t1 - t0; out[1] = sink; }
  tc::tc_fence_before();
  __syncthreads();
  if (warp == 0) { tc::tc_fence_after(); tc::tmem_dealloc(tmem_base_s, 512); }
}

// fp64: chains of independent DFMA / DMMA (mma.sync.m8n8k4.f64) per warp, 8 warps
__global__ void __launch_bounds__(256, 1) fp64_kernel(int use_dmma, long long* out, double* sink) {
  double c[8][2], a = 1.0 + threadIdx.x * 1e-9, b = 1.0 - threadIdx.x * 1e-9;
#pragma unroll
  for (int i = 0; i < 8; ++i) { c[i][0] = i; c[i][1] = -i; }
  __syncthreads();
  const long long t0 = clock64();
  for (int r = 0; r < REPS; ++r) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      if (use_dmma)
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
      else { c[i][0] = fma(a, b, c[i][0]); c[i][1] = fma(a, b, c[i][1]); }
    }
  }
  __syncthreads();
  const long long t1 = clock64();
  double s = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1];
  if (threadIdx.x == 0) out[0] = t1 - t0;
  sink[threadIdx.x] = s;
}

}  // namespace

int main() {
  long long* d_out; double* d_sink;
  cudaMalloc(&d_out, 64); cudaMalloc(&d_sink, 256 * 8);
  long long h[2];
  cudaFuncSetAttribute(mma_i8_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 66 * 1024);
  cudaFuncSetAttribute(mma_i8_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 66 * 1024);
  cudaFuncSetAttribute(mma_i8_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, 66 * 1024);
  printf("| N | K-major no swizzle, aligned | no swizzle, start shifted one row | 64-byte swizzle | 128-byte swizzle | tensor-pipe time N/2 | operand-fetch model 32 + N/4 |\n|---|---|---|---|---|---|---|\n");
  const int Ns[] = {16, 32, 48, 64, 96, 128, 192, 256};
  for (int N : Ns) {
    printf("| %d |", N);
    const int layouts[] = {0, 1, 4, 2};
    for (int L : layouts) {
      mma_i8_kernel<1><<<1, 128, 66 * 1024>>>(N, L, d_out);
      if (cudaDeviceSynchronize() != cudaSuccess) { printf(" error |"); continue; }
      cudaMemcpy(h, d_out, 8, cudaMemcpyDeviceToHost);
      printf(" %.1f |", (double)h[0] / REPS);
    }
    printf(" %d | %d |\n", N / 2, 32 + N / 4);
  }
  printf("\nclk per tcgen05.mma kind::i8 (M = 128, K = 32 bytes), %d back-to-back MMAs into one accumulator, one CTA.\n\n", REPS);
  printf("| N | one accumulator | rotating over 2 accumulators | rotating over 4 (N <= 128) |\n|---|---|---|---|\n");
  for (int N : Ns) {
    printf("| %d |", N);
    for (int na = 1; na <= 4; na *= 2) {
      if (na * N > 512) { printf(" - |"); continue; }
      if (na == 1) mma_i8_kernel<1><<<1, 128, 66 * 1024>>>(N, 4, d_out);
      else if (na == 2) mma_i8_kernel<2><<<1, 128, 66 * 1024>>>(N, 4, d_out);
      else mma_i8_kernel<4><<<1, 128, 66 * 1024>>>(N, 4, d_out);
      if (cudaDeviceSynchronize() != cudaSuccess) { printf(" error |"); continue; }
      cudaMemcpy(h, d_out, 8, cudaMemcpyDeviceToHost);
      printf(" %.1f |", (double)h[0] / REPS);
    }
    printf("\n");
  }
  printf("\nsame chain, 64-byte swizzle, the destination rotating over several accumulators: is the 32 + N/4 floor a dependency on the accumulator?\n\n");
  printf("| tcgen05.ld 32x32b.x16 | clk per load, 4 warps | 8 warps | 16 warps | bytes/clk/SM at 16 warps |\n|---|---|---|---|---|\n");
  for (int inflight = 1; inflight <= 4; inflight *= 2) {
    printf("| %d in flight per wait |", inflight);
    double last = 0;
    for (int nw = 4; nw <= 16; nw *= 2) {
      tmem_ld_kernel<<<1, nw * 32>>>(inflight, d_out);
      cudaDeviceSynchronize();
      cudaMemcpy(h, d_out, 8, cudaMemcpyDeviceToHost);
      last = (double)h[0] / REPS;
      printf(" %.1f |", last);
    }
    printf(" %.0f |\n", 16.0 * 32 * 16 * 4 / last);
  }
  printf("\n| fp64 | FMA/clk/SM (8 warps, 8 independent chains each) |\n|---|---|\n");
  for (int dm = 0; dm <= 1; ++dm) {
    fp64_kernel<<<1, 256>>>(dm, d_out, d_sink);
    cudaDeviceSynchronize();
    cudaMemcpy(h, d_out, 8, cudaMemcpyDeviceToHost);
    const double fma_per = dm ? 8.0 * 8 * 8 * 4 * 8 : 256.0 * 16;      // per iteration: DMMA 8x8x4 = 256 FMA per warp-instruction
    printf("| %s | %.1f |\n", dm ? "DMMA mma.sync.m8n8k4.f64" : "DFMA", fma_per * REPS / (double)h[0]);
  }
  return 0;
}
