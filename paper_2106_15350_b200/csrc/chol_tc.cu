// chol_tc.cu -- K3 on the tensor pipe: the trailing updates of the blocked Cholesky (F3, PAPER.md:70-74
// `cp.linalg.solve`) as int8 digit products on tcgen05 with int32 TMEM accumulators.
//
// A right-looking blocked Cholesky spends dim^3/3 of its dim^3/3 + O(dim^2 nb) flops in
//     A22 <- A22 - P P^T,        P = the finished panel rows  L[r0.., k0..k0+K)   (fp64, K = 64 .. 1024 columns).
// The fp64 pipe (DMMA, 37 TFLOP/s) caps that at >= 158 ms for the 32 systems of 8192 of configs[4]; the int8 tensor
// pipe is ~100x wider.  P is therefore quantised row by row (Ozaki-style error-free slicing):
//     q[i][k] = rint(P[i][k] * 2^(30 - e_i)),   2^(e_i - 1) <= max_k |P[i][k]| < 2^e_i      (|q| <= 2^30)
//     q = d0 + 256 d1 + 256^2 d2 + 256^3 d3,    d in [-128, 127]   (four balanced radix-256 digits)
// and   sum_k q[i][k] q[j][k] = sum_s 256^s T_s,   T_s = sum_{a+b=s} sum_k d_a[i][k] d_b[j][k]   (int8 x int8 -> int32, exact).
// Only the diagonals s = 3..6 are issued (10 of the 16 digit products): the dropped ones are below 2^-27 of the
// product of the two row maxima, the same order as the rounding of q (2^-31 per factor).  That is ~2^-27 relative
// backward error per update against 2^-53 for fp64 and 2^-24 for an fp32 factorisation -- SURVEY.md Appendix A: W error
// ~ 4e3 x elementwise perturbation, so ~3e-5 of the 1e-3 budget, and no refinement sweep is needed.  The matrix itself
// stays in fp64 (read-modify-write in the epilogue), the diagonal blocks and the panel solves stay on the fp64 path.
//
// Pipeline (one CTA per 128 x 128 tile of the update region, tiles above the diagonal skipped):
//   panel_split_kernel : fp64 panel rows -> digit planes int8 [cand][4][row][pitch] (K contiguous) + row scales
//   warp 0             : TMA producer, 64-byte K chunks, 64-byte swizzle, 3-stage mbarrier ring (8 tiles of 8 KB per stage)
//   warp 1             : one thread issues tcgen05.mma kind::i8 (M = 128, N = 128, K = 32), K-major operands
//   warps 2..9         : epilogue: tcgen05.ld the four diagonals, int64 recombination, scale, A -= (fp64 RMW)
#include "internal.h"
#include "tc_common.cuh"
#include <cuda.h>

namespace {

constexpr int ND = 4;                    // digits per entry
constexpr int TM = 128, TN = 128;        // output tile = UMMA M x N
constexpr int KC = 64;                   // K bytes per pipeline stage = one 64-byte swizzle row (two K = 32 MMA steps)
constexpr int ATILE = TM * KC, BTILE = TN * KC;
constexpr int STAGE_BYTES = ND * (ATILE + BTILE);      // 64 KB
constexpr int NSTAGE = 3;
constexpr int NTHREADS = 320;            // producer, issuer, 8 epilogue warps
constexpr int TMEM_COLS = 512;           // 4 diagonals x 128 columns
constexpr uint32_t LAYOUT_SW64 = 4;

struct SyrkParams {
  double* A; long long a_stride, ld;
  const double* rscale;                  // [n_cand][rows]: 2^(e_i - 30 + 12)
  long long rows, dim;                   // rows = dim + appended right-hand-side rows
  int r0, c0, c1;                        // update rows [r0, rows) x columns [c0, c1), lower triangle inside [0, dim)
  int n_iters;                           // K / 64
  unsigned long long* ops;               // int8 multiply-adds issued (measurement; may be NULL)
};

// one warp per row: scale from the row maximum, four balanced digits, zero padding up to Kp
__global__ void __launch_bounds__(256) panel_split_kernel(const double* __restrict__ A, long long a_stride, long long ld,
                                                          long long rows, int r0, int k0, int K, int Kp, int pitch,
                                                          int8_t* __restrict__ planes, double* __restrict__ rscale) {
  const long long z = blockIdx.y;
  const long long i = r0 + (long long)blockIdx.x * 8 + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (i >= rows) return;
  const double* src = A + z * a_stride + i * ld + k0;
  double mx = 0.0;
  for (int k = lane; k < K; k += 32) mx = fmax(mx, fabs(src[k]));
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, d));
  int e = 0;
  if (mx > 0.0 && mx < 1.0e300) frexp(mx, &e);               // mx = m 2^e, m in [0.5, 1)
  const double up = scalbn(1.0, 30 - e);
  if (lane == 0) rscale[z * rows + i] = scalbn(1.0, e - 30 + 12);
  const long long plane = rows * (long long)pitch;
  int8_t* dst = planes + (z * ND * rows + i) * pitch;
  for (int g = lane * 4; g < Kp; g += 128) {
    uint32_t w[ND] = {0u, 0u, 0u, 0u};
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      const int k = g + t;
      int v = (k < K) ? __double2int_rn(src[k] * up) : 0;
#pragma unroll
      for (int a = 0; a < ND; ++a) {
        const int d = (int)(int8_t)(v & 0xFF);
        w[a] |= (uint32_t)(d & 0xFF) << (8 * t);
        v = (v - d) >> 8;
      }
    }
#pragma unroll
    for (int a = 0; a < ND; ++a) *reinterpret_cast<uint32_t*>(dst + a * plane + g) = w[a];
  }
}

__global__ void __launch_bounds__(NTHREADS, 1) syrk_tc_kernel(const __grid_constant__ CUtensorMap tmap, const SyrkParams p) {
  const int tj = blockIdx.x, ti = blockIdx.y, z = blockIdx.z;
  const int i0 = p.r0 + ti * TM, j0 = p.c0 + tj * TN;
  if (i0 + TM - 1 < p.dim && j0 > i0 + TM - 1) return;      // every row of the tile lies in the square part, above the diagonal
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t bar_full[NSTAGE], bar_empty[NSTAGE], bar_tmem;
  __shared__ uint32_t tmem_base_s;
  const int warp = tc::uniform_warp_id(), lane = threadIdx.x & 31;
  const uint32_t smem0 = tc::smem_u32(smem);

  if (warp == 0 && lane == 0) {
    tc::prefetch_tensormap(&tmap);
    for (int s = 0; s < NSTAGE; ++s) { tc::mbar_init(tc::smem_u32(&bar_full[s]), 1); tc::mbar_init(tc::smem_u32(&bar_empty[s]), 1); }
    tc::mbar_init(tc::smem_u32(&bar_tmem), 1);
    tc::fence_barrier_init();
  }
  if (warp == 1) tc::tmem_alloc(tc::smem_u32(&tmem_base_s), TMEM_COLS);
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t tmem = tmem_base_s;

  if (warp == 0) {
    // ===== TMA producer =====
    int s = 0, ph = 0;
    for (int it = 0; it < p.n_iters; ++it) {
      tc::mbar_wait(tc::smem_u32(&bar_empty[s]), ph ^ 1);
      if (tc::elect_one()) {
        const uint32_t full = tc::smem_u32(&bar_full[s]);
        tc::mbar_arrive_expect_tx(full, STAGE_BYTES);
        const uint32_t base = smem0 + s * STAGE_BYTES;
#pragma unroll
        for (int a = 0; a < ND; ++a) {
          tc::tma_load_3d(base + a * ATILE, &tmap, full, it * KC, i0, z * ND + a);
          tc::tma_load_3d(base + ND * ATILE + a * BTILE, &tmap, full, it * KC, j0, z * ND + a);
        }
      }
      __syncwarp();
      if (++s == NSTAGE) { s = 0; ph ^= 1; }
    }
  } else if (warp == 1) {
    // ===== MMA issuer: diagonals s = a + b = 3..6 into accumulators 0..3 =====
    constexpr uint32_t idesc = tc::idesc_i8(TM, TN, 1, 1, 0, 0);
    const uint64_t d0 = tc::smem_desc(smem0, 16, 8 * KC, LAYOUT_SW64);
    int s = 0, ph = 0;
    for (int it = 0; it < p.n_iters; ++it) {
      tc::mbar_wait(tc::smem_u32(&bar_full[s]), ph);
      tc::tc_fence_after();
      const uint64_t ds = d0 + (uint64_t)(s * (STAGE_BYTES >> 4));
#pragma unroll
      for (int kk = 0; kk < KC / 32; ++kk) {
#pragma unroll
        for (int sd = ND - 1; sd <= 2 * (ND - 1); ++sd) {
#pragma unroll
          for (int a = 0; a < ND; ++a) {
            const int b = sd - a;
            if (b >= 0 && b < ND) {
              const uint64_t da = ds + (uint64_t)((a * ATILE + kk * 32) >> 4);
              const uint64_t db = ds + (uint64_t)((ND * ATILE + b * BTILE + kk * 32) >> 4);
              const bool first = (kk == 0) && (a == sd - (ND - 1));      // smallest a of this diagonal
              if (tc::elect_one()) tc::mma_i8(tmem + (sd - (ND - 1)) * TN, da, db, idesc, (first && it == 0) ? 0u : 1u);
            }
          }
        }
      }
      if (tc::elect_one()) tc::mma_commit(tc::smem_u32(&bar_empty[s]));
      __syncwarp();
      if (++s == NSTAGE) { s = 0; ph ^= 1; }
    }
    if (tc::elect_one()) {
      tc::mma_commit(tc::smem_u32(&bar_tmem));
      if (p.ops) atomicAdd(p.ops, (unsigned long long)p.n_iters * (KC / 32) * 10ull * (TM * TN * 32));
    }
    __syncwarp();
  } else {
    // ===== epilogue: warp w owns TMEM lanes 32 (w % 4) .. +31 and 64 of the 128 columns =====
    // Phase 1: accumulators -> scaled fp64 update values -> shared memory (the operand ring is idle once bar_tmem has
    // fired: every MMA, hence every read of it, has completed).  Phase 2: each warp walks whole rows with the lanes
    // across the columns, so the read-modify-write of A is coalesced (a thread per row would touch 32 rows
    // ld * 8 bytes apart per access -- with ld = 8192 every one of them in the same L2 set).
    const int q = warp & 3, ew = warp - 2, half = ew >> 2;
    double* S = reinterpret_cast<double*>(smem);                 // [TM][SP]
    constexpr int SP = TN + 1;
    tc::mbar_wait(tc::smem_u32(&bar_tmem), 0);
    tc::tc_fence_after();
    const double* rs = p.rscale + (long long)z * p.rows;
    {
      const int r = q * 32 + lane;
      const long long i = (long long)i0 + r;
      const double ri = (i < p.rows) ? rs[i] : 0.0;
      for (int c0 = half * 64; c0 < half * 64 + 64; c0 += 16) {
        uint32_t acc[ND][16];
#pragma unroll
        for (int s = 0; s < ND; ++s) tc::tmem_ld16(tmem + ((uint32_t)(q * 32) << 16) + s * TN + c0, acc[s]);
        tc::tmem_ld_wait();
#pragma unroll
        for (int e = 0; e < 16; ++e) {
          long long g = 0;
#pragma unroll
          for (int s = ND - 1; s >= 0; --s) g = g * 256 + (long long)(int32_t)acc[s][e];
          const long long j = (long long)j0 + c0 + e;
          S[r * SP + c0 + e] = (double)g * (ri * ((j < p.c1) ? rs[j] : 0.0));
        }
      }
    }
    asm volatile("bar.sync 1, 256;" ::: "memory");                // the eight epilogue warps
    // 8 rows x 128 columns per batch: all 32 loads of a lane are issued before the first subtract, so a warp keeps
    // 8 KB in flight (the per-SM share of HBM needs tens of KB in flight; a load-subtract-store chain per row does not)
#pragma unroll 1
    for (int rb = 0; rb < TM / 8; rb += 8) {
      double v[8][TN / 32];
#pragma unroll
      for (int rr = 0; rr < 8; ++rr) {
        const int r = ew * (TM / 8) + rb + rr;
        const long long i = (long long)i0 + r;
        const long long jmax = (i < p.dim) ? i : (long long)p.c1 - 1;      // last column this row stores
        const double* Arow = p.A + (long long)z * p.a_stride + i * p.ld;
#pragma unroll
        for (int t = 0; t < TN / 32; ++t) {
          const long long j = (long long)j0 + lane + 32 * t;
          v[rr][t] = (i < p.rows && j < p.c1 && j <= jmax) ? __ldcs(Arow + j) : 0.0;
        }
      }
#pragma unroll
      for (int rr = 0; rr < 8; ++rr) {
        const int r = ew * (TM / 8) + rb + rr;
        const long long i = (long long)i0 + r;
        const long long jmax = (i < p.dim) ? i : (long long)p.c1 - 1;
        double* Arow = p.A + (long long)z * p.a_stride + i * p.ld;
#pragma unroll
        for (int t = 0; t < TN / 32; ++t) {
          const long long j = (long long)j0 + lane + 32 * t;
          if (i < p.rows && j < p.c1 && j <= jmax) Arow[j] = v[rr][t] - S[r * SP + lane + 32 * t];
        }
      }
    }
    tc::tc_fence_before();
  }
  __syncthreads();
  if (warp == 1) { tc::tc_fence_after(); tc::tmem_dealloc(tmem, TMEM_COLS); }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn get_encode() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  return fn;
}

}  // namespace

// scratch: digit planes [n_cand][4][rows][pitch] + row scales [n_cand][rows]
size_t lb_chol_tc_ws_bytes(int64_t rows, int n_cand, int kmax) {
  const int64_t pitch = lb_align_up(kmax, KC);
  return (size_t)lb_align_up((int64_t)n_cand * ND * rows * pitch, 256) + (size_t)lb_align_up((int64_t)n_cand * rows * 8, 256);
}

int lb_chol_tc_begin(lbcnn_handle_s* h, void* ws, int64_t rows, int64_t dim, int n_cand, int kmax, double* A,
                     long long a_stride, long long ld, unsigned long long* ops, CholTcCtx* ctx) {
  EncodeTiledFn enc = get_encode();
  if (!enc) return LBCNN_ERR_CUDA;
  const int64_t pitch = lb_align_up(kmax, KC);
  ctx->planes = reinterpret_cast<int8_t*>(ws);
  ctx->rscale = reinterpret_cast<double*>(reinterpret_cast<char*>(ws) + lb_align_up((int64_t)n_cand * ND * rows * pitch, 256));
  ctx->pitch = (int)pitch; ctx->rows = rows; ctx->dim = dim; ctx->n_cand = n_cand;
  ctx->A = A; ctx->a_stride = a_stride; ctx->ld = ld; ctx->ops = ops;
  static_assert(sizeof(ctx->tmap) >= sizeof(CUtensorMap), "tensor map storage");
  const cuuint64_t gdim[3] = {(cuuint64_t)pitch, (cuuint64_t)rows, (cuuint64_t)n_cand * ND};
  const cuuint64_t gstr[2] = {(cuuint64_t)pitch, (cuuint64_t)rows * pitch};
  const cuuint32_t box[3] = {KC, TM, 1};
  const cuuint32_t estr[3] = {1, 1, 1};
  if (enc(reinterpret_cast<CUtensorMap*>(ctx->tmap), CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, ctx->planes, gdim, gstr, box, estr,
          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
    return LBCNN_ERR_CUDA;
  const size_t smem = (size_t)NSTAGE * STAGE_BYTES + 1024;
  LB_CUDA_OK(cudaFuncSetAttribute(syrk_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  (void)h;
  return LBCNN_OK;
}

// A[i][j] -= sum_{k in [k0, k0 + K)} L[i][k] L[j][k]   for i in [r0, rows), j in [r0, c1), j <= i when i < dim
int lb_chol_tc_update(lbcnn_handle_s* h, const CholTcCtx& ctx, int r0, int c1, int k0, int K, cudaStream_t st) {
  if (ctx.rows - r0 <= 0 || c1 - r0 <= 0 || K <= 0) return LBCNN_OK;
  if (K > ctx.pitch) return LBCNN_ERR_INVALID_ARG;
  const int Kp = (int)lb_align_up(K, KC);
  dim3 gs((unsigned)((ctx.rows - r0 + 7) / 8), (unsigned)ctx.n_cand);
  panel_split_kernel<<<gs, 256, 0, st>>>(ctx.A, ctx.a_stride, ctx.ld, ctx.rows, r0, k0, K, Kp, ctx.pitch, ctx.planes, ctx.rscale);
  h->launches += 1;
  SyrkParams p{};
  p.A = ctx.A; p.a_stride = ctx.a_stride; p.ld = ctx.ld; p.rscale = ctx.rscale; p.rows = ctx.rows; p.dim = ctx.dim;
  p.r0 = r0; p.c0 = r0; p.c1 = c1; p.n_iters = Kp / KC; p.ops = ctx.ops;
  dim3 grid((unsigned)((c1 - r0 + TN - 1) / TN), (unsigned)((ctx.rows - r0 + TM - 1) / TM), (unsigned)ctx.n_cand);
  const size_t smem = (size_t)NSTAGE * STAGE_BYTES + 1024;
  syrk_tc_kernel<<<grid, NTHREADS, smem, st>>>(*reinterpret_cast<const CUtensorMap*>(ctx.tmap), p);
  h->launches += 1;
  LB_CUDA_OK(cudaGetLastError());
  return LBCNN_OK;
}
