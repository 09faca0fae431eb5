// gram_tc.cu -- K2 on the tensor pipe: the EXACT Gram matrix of integer-valued features (F1, PAPER.md:66-70
// `cp.dot(H,H.T)`), A = U^T U + lam I, with tcgen05.mma kind::i8 and int32 accumulators in TMEM.
//
// The expander's features are exact integers (R14).  Every integer u with |u| <= 8355711 is written
// as balanced radix-256 digits  u = d0 + 256 d1 + 65536 d2,  d in [-128, 127]  (1, 2 or 3 digits, chosen
// per candidate from the data), so
//     G[i][j] = sum_n u[n][i] u[n][j] = sum_s 256^s P_s[i][j],   P_s = sum_{a+b=s} D_a^T D_b
// where every P_s is a sum of int8 x int8 products: exact in the tensor core's int32 accumulators as long as
// 3 * 128^2 * n < 2^31, i.e. n <= 43690 samples (larger n takes the fp64 SIMT path).  The epilogue
// recombines the P_s in int64 and rounds ONCE to fp64 -- the Gram is bit-exact, which is what the
// conditioning of the configs' systems needs (cond ~ 1e6; an fp32-accumulated Gram misses the 1e-3
// tolerance on W).  9 int8 MMAs (3 digits) cost 2.25 TF32-MMA equivalents, 4 (2 digits)
// cost 1 -- cheaper than 3xTF32 and exact.
//
// Pipeline (one CTA per 128 x 96 output tile of one candidate, lower-triangle tiles only):
//   split kernel : fp32 H [K][n][F] -> digit planes int8 [K][3][n][Fp] (F contiguous) + digits needed per candidate
//   warp 0       : TMA producer, 64-sample stages of the digit planes (128-byte swizzle), mbarrier ring
//   warp 1       : one thread issues tcgen05.mma (M=128, N=96, K=32; MN-major operands: the feature index
//                  is contiguous in memory, no transpose anywhere); tcgen05.commit frees stages
//   warps 2..5   : epilogue, tcgen05.ld the 2L-1 accumulators, int64 recombination, fp64 store
#include "internal.h"
#include "tc_common.cuh"
#include <cuda.h>

namespace {

constexpr int TM = 128;        // output tile rows (features i)   = UMMA M
constexpr int TN = 96;         // output tile columns (features j) = UMMA N
constexpr int KS = 64;         // samples per pipeline stage (two K = 32 MMA steps)
constexpr int BOXW = 128;      // TMA box width in features (= bytes): one 128-byte swizzle row
constexpr int TILE_BYTES = KS * BOXW;          // 8 KB per digit plane per operand per stage
constexpr int RING_BYTES = 24 * TILE_BYTES;   // 192 KB of operand stages: 12 / 6 / 4 stages for 1 / 2 / 3 digits
constexpr int MAXSTAGE = 12;
constexpr int TMEM_COLS = 512; // 5 accumulators x 96 columns = 480
constexpr int NTHREADS = 192;

struct GramTcParams {
  const int32_t* nlimb;   // [n_cand] digits needed (1..3)
  const int32_t* nl32;    // [n_cand][G32] digits needed per group of 32 features (primal: per-tile digit counts)
  int G32;
  double* A; long long a_stride, ld;
  int F, n, n_iters;   // F = dimension of the OUTPUT matrix (features, or samples in the dual branch)
  int Fcols;           // columns written (primal with fused right-hand side: F features of F + c output rows)
  int dual;            // 0: A = U^T U (operands MN-major: the feature index is contiguous); 1: A = U U^T (K-major)
  double lam;
  unsigned long long* ops;   // int8 multiply-adds issued (measurement)
  int accumulate;            // A += G (a further chunk of samples of a streamed Gram) instead of A = G
  int rshift;                // output rows >= Fcols are stored rshift rows further down (dual: cross-Gram rows behind the right-hand sides)
  int add_lam;               // ... + lam I (the last chunk: (G1 + G2 + ..) + lam rounds like the unstreamed G + lam)
};

// ---- digit split ----------------------------------------------------------------------------------
// Balanced radix-256 digits without branches: d0 = low byte of u (as int8), d1 = byte 1 of u + 128, d2 = byte 2 of
// u + 128 + 32768 (the carries of the balanced representation are exactly those two additions); a second digit
// is needed iff (u + 128) >> 8 != 0, a third iff (u + 32896) >> 16 != 0.  A thread converts 8 consecutive
// features of one sample (two float4 loads) and writes 8 bytes per plane; byte packing is three PRMTs per word.
__device__ __forceinline__ uint32_t pack_bytes(uint32_t a, uint32_t b, uint32_t c, uint32_t d, uint32_t sel) {
  // byte `sel` (0..2) of a, b, c, d -> one word
  const uint32_t s2 = sel | ((sel + 4) << 4);
  return __byte_perm(__byte_perm(a, b, s2), __byte_perm(c, d, s2), 0x5410);
}
__global__ void __launch_bounds__(256) split_kernel(const float* __restrict__ U, long long n, int F, int Fp,
                                                    int8_t* __restrict__ planes, int32_t* __restrict__ nlimb,
                                                    int32_t* __restrict__ nl32, int G32, int32_t* __restrict__ info,
                                                    const int32_t* __restrict__ y, int c_aug) {
  const int z = blockIdx.y;
  const long long oct_per_row = Fp / 8;
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  uint32_t or2 = 0, or3 = 0;
  bool bad = false;          // a value outside the three-digit envelope, or not an integer: the LBCNN_H_INTEGER promise is broken
  if (t < n * oct_per_row) {
    const long long row = t / oct_per_row;
    const int f0 = (int)(t % oct_per_row) * 8;
    const float* src = U + ((long long)z * n + row) * F + f0;
    int v[8];
    if ((F & 3) == 0 && f0 + 8 <= F) {
      const float4 x = __ldcs(reinterpret_cast<const float4*>(src));
      const float4 y = __ldcs(reinterpret_cast<const float4*>(src) + 1);
      v[0] = (int)x.x; v[1] = (int)x.y; v[2] = (int)x.z; v[3] = (int)x.w;
      v[4] = (int)y.x; v[5] = (int)y.y; v[6] = (int)y.z; v[7] = (int)y.w;
      bad = !((float)v[0] == x.x && (float)v[1] == x.y && (float)v[2] == x.z && (float)v[3] == x.w &&
              (float)v[4] == y.x && (float)v[5] == y.y && (float)v[6] == y.z && (float)v[7] == y.w);
    } else {
#pragma unroll
      // columns F .. F + c_aug - 1 of plane 0: the one-hot coding of the sample's label (fused right-hand side)
      const int lab = c_aug ? y[row] : -1;
      for (int q = 0; q < 8; ++q) {
        const float x = (f0 + q < F) ? src[q] : ((f0 + q - F == lab && lab < c_aug) ? 1.0f : 0.0f);
        v[q] = (int)x;
        bad = bad || !((float)v[q] == x);
      }
    }
    uint32_t t1[8], t2[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      t1[q] = (uint32_t)(v[q] + 128);
      t2[q] = (uint32_t)(v[q] + 32896);
      or2 |= t1[q] & 0xFFFFFF00u;
      or3 |= t2[q] & 0xFFFF0000u;
      bad = bad || (t2[q] + 0x800000u) >= 0x1000000u;       // third digit (t2 >> 16) outside [-128, 127]
    }
    if (bad) info[z] = -1;
    uint2 w0, w1, w2;
    w0.x = pack_bytes((uint32_t)v[0], (uint32_t)v[1], (uint32_t)v[2], (uint32_t)v[3], 0);
    w0.y = pack_bytes((uint32_t)v[4], (uint32_t)v[5], (uint32_t)v[6], (uint32_t)v[7], 0);
    w1.x = pack_bytes(t1[0], t1[1], t1[2], t1[3], 1);
    w1.y = pack_bytes(t1[4], t1[5], t1[6], t1[7], 1);
    w2.x = pack_bytes(t2[0], t2[1], t2[2], t2[3], 2);
    w2.y = pack_bytes(t2[4], t2[5], t2[6], t2[7], 2);
    int8_t* dst = planes + ((long long)z * 3 * n + row) * Fp + f0;
    const long long plane = n * (long long)Fp;
    *reinterpret_cast<uint2*>(dst) = w0;
    *reinterpret_cast<uint2*>(dst + plane) = w1;
    *reinterpret_cast<uint2*>(dst + 2 * plane) = w2;
  }
  int need = or3 ? 3 : (or2 ? 2 : 1);
  // digits needed by this thread's group of 32 features (very few values need the third digit, so most 128 x 96 tiles
  // of the Gram run with 2 x 2 instead of 3 x 3 digit products); same cached-read trick as below
  if (need > 1 && t < n * oct_per_row) {
    int32_t* g = nl32 + (long long)z * G32 + (int)((t % oct_per_row) >> 2);
    if (need > __ldg(g)) atomicMax(g, need);     // a stale (smaller) cached value only costs one redundant atomic
  }
  need = __reduce_max_sync(0xffffffffu, need);
  // one atomic per warp only while it can still raise the count: after the first few warps of a candidate the
  // (L2-cached) read already shows the final value and no further atomics reach that address
  if ((threadIdx.x & 31) == 0 && need > 1 && need > *reinterpret_cast<volatile int32_t*>(&nlimb[z])) atomicMax(&nlimb[z], need);
}

// digit counts = 1 and (zero != NULL) the candidates' info words = 0, in one launch
__global__ void fill_i32_kernel(int32_t* p, int n, int32_t v, int32_t* zero, int nz) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t < n) p[t] = v;
  if (zero && t < nz) zero[t] = 0;
}

// ---- the Gram kernel ------------------------------------------------------------------------------
// Role loops run warp-uniformly (uniform_warp_id) and are specialised on the digit count L, so every stage / plane /
// K-step offset is a compile-time constant and a descriptor is "base + constant": the issuing warp spends a few
// uniform-datapath instructions per MMA instead of rebuilding descriptors in vector registers (which cost ~150 clk
// per MMA, three times the MMA itself).
// Dual branch (A = U U^T, F >= n): the contraction runs over the contiguous feature index, so the operands are
// K-major 128-byte-swizzled tiles [128 or 96 samples][128 features]; a stage holds 128 features (four K = 32 steps).
constexpr int DTILE_A = TM * 128, DTILE_B = TN * 128;
template <int L, bool DUAL> struct GramCfg {
  static constexpr int STAGE_BYTES = DUAL ? L * (DTILE_A + DTILE_B) : 2 * L * TILE_BYTES;
  static constexpr int NSTAGE = (RING_BYTES / STAGE_BYTES) > MAXSTAGE ? MAXSTAGE : (RING_BYTES / STAGE_BYTES);
};

template <int L, bool DUAL>
__device__ __forceinline__ void gram_produce(const CUtensorMap* tmap, const CUtensorMap* tmapB, const GramTcParams& p, uint32_t smem0,
                                             uint64_t* bar_full, uint64_t* bar_empty, int i0, int j0, int z) {
  constexpr int NSTAGE = GramCfg<L, DUAL>::NSTAGE, STAGE_BYTES = GramCfg<L, DUAL>::STAGE_BYTES;
  int s = 0, ph = 0;
  for (int it = 0; it < p.n_iters; ++it) {
    tc::mbar_wait(tc::smem_u32(&bar_empty[s]), ph ^ 1);
    if (tc::elect_one()) {
      const uint32_t full = tc::smem_u32(&bar_full[s]);
      tc::mbar_arrive_expect_tx(full, STAGE_BYTES);
      const uint32_t base = smem0 + s * STAGE_BYTES;
#pragma unroll
      for (int a = 0; a < L; ++a) {
        if (DUAL) {
          tc::tma_load_3d(base + a * DTILE_A, tmap, full, it * 128, i0, z * 3 + a);
          tc::tma_load_3d(base + L * DTILE_A + a * DTILE_B, tmapB, full, it * 128, j0, z * 3 + a);
        } else {
          tc::tma_load_3d(base + a * TILE_BYTES, tmap, full, i0, it * KS, z * 3 + a);
          tc::tma_load_3d(base + (L + a) * TILE_BYTES, tmap, full, j0, it * KS, z * 3 + a);
        }
      }
    }
    __syncwarp();
    if (++s == NSTAGE) { s = 0; ph ^= 1; }
  }
}

template <int L, bool DUAL>
__device__ __forceinline__ void gram_issue(const GramTcParams& p, uint32_t smem0, uint32_t tmem, uint64_t* bar_full,
                                           uint64_t* bar_empty, uint64_t* bar_tmem) {
  constexpr int NSTAGE = GramCfg<L, DUAL>::NSTAGE, STAGE_BYTES = GramCfg<L, DUAL>::STAGE_BYTES;
  constexpr uint32_t idesc = DUAL ? tc::idesc_i8(TM, TN, 1, 1, 0, 0) : tc::idesc_i8(TM, TN, 1, 1, 1, 1);
  constexpr int KSTEPS = DUAL ? 4 : KS / 32;
  // descriptor of the ring's first byte; every operand is this plus a constant number of 16-byte units
  // (K-major swizzled tiles: 8-row groups 1024 B apart, a K = 32 step is 32 bytes inside the 128-byte row)
  const uint64_t d0 = DUAL ? tc::smem_desc(smem0, 16, 1024, tc::LAYOUT_SW128) : tc::smem_desc(smem0, TILE_BYTES, 8 * BOXW, tc::LAYOUT_SW128);
  int s = 0, ph = 0;
  for (int it = 0; it < p.n_iters; ++it) {
    tc::mbar_wait(tc::smem_u32(&bar_full[s]), ph);
    tc::tc_fence_after();
    const uint64_t ds = d0 + (uint64_t)(s * (STAGE_BYTES >> 4));
#pragma unroll
    for (int kk = 0; kk < KSTEPS; ++kk) {
#pragma unroll
      for (int a = 0; a < L; ++a) {
#pragma unroll
        for (int b = 0; b < L; ++b) {
          const uint64_t da = ds + (uint64_t)((DUAL ? a * DTILE_A + kk * 32 : a * TILE_BYTES + kk * 32 * BOXW) >> 4);
          const uint64_t db = ds + (uint64_t)((DUAL ? L * DTILE_A + b * DTILE_B + kk * 32 : (L + b) * TILE_BYTES + kk * 32 * BOXW) >> 4);
          // accumulator a + b; its first product of the whole tile is (a, b) with a = max(0, a + b - L + 1) at it = kk = 0
          const bool first = (kk == 0) && (a == ((a + b) > (L - 1) ? (a + b) - (L - 1) : 0));
          if (tc::elect_one()) tc::mma_i8(tmem + (a + b) * TN, da, db, idesc, (first && it == 0) ? 0u : 1u);
        }
      }
    }
    if (tc::elect_one()) tc::mma_commit(tc::smem_u32(&bar_empty[s]));     // stage free once these MMAs have read it
    __syncwarp();
    if (++s == NSTAGE) { s = 0; ph ^= 1; }
  }
  if (tc::elect_one()) tc::mma_commit(tc::smem_u32(bar_tmem));             // accumulators complete
  __syncwarp();
}

// Primal branch with per-tile digit counts: the row tile needs Li digits, the column tile Lj (from the 32-feature
// group counts), so only Li x Lj of the nine digit products are issued and only Li + Lj planes are loaded.  Stage =
// Li + Lj tile slots of 8 KB (A planes, then B planes); as many stages as fit the 192 KB ring (at most 12).
__device__ __forceinline__ void gram_produce_p(const CUtensorMap* tmap, const GramTcParams& p, uint32_t smem0, uint64_t* bar_full,
                                               uint64_t* bar_empty, int i0, int j0, int z, int Li, int Lj) {
  int s = 0, ph = 0;
  const uint32_t tx_bytes = (uint32_t)(Li + Lj) * TILE_BYTES;
  const int PSTAGE_BYTES = (Li + Lj) * TILE_BYTES, PNSTAGE = min(MAXSTAGE, 24 / (Li + Lj));
  for (int it = 0; it < p.n_iters; ++it) {
    tc::mbar_wait(tc::smem_u32(&bar_empty[s]), ph ^ 1);
    if (tc::elect_one()) {
      const uint32_t full = tc::smem_u32(&bar_full[s]);
      tc::mbar_arrive_expect_tx(full, tx_bytes);
      const uint32_t base = smem0 + s * PSTAGE_BYTES;
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        if (a < Li) tc::tma_load_3d(base + a * TILE_BYTES, tmap, full, i0, it * KS, z * 3 + a);
        if (a < Lj) tc::tma_load_3d(base + (Li + a) * TILE_BYTES, tmap, full, j0, it * KS, z * 3 + a);
      }
    }
    __syncwarp();
    if (++s == PNSTAGE) { s = 0; ph ^= 1; }
  }
}

__device__ __forceinline__ void gram_issue_p(const GramTcParams& p, uint32_t smem0, uint32_t tmem, uint64_t* bar_full,
                                             uint64_t* bar_empty, uint64_t* bar_tmem, int Li, int Lj) {
  constexpr uint32_t idesc = tc::idesc_i8(TM, TN, 1, 1, 1, 1);
  const uint64_t d0 = tc::smem_desc(smem0, TILE_BYTES, 8 * BOXW, tc::LAYOUT_SW128);
  const int PSTAGE_BYTES = (Li + Lj) * TILE_BYTES, PNSTAGE = min(MAXSTAGE, 24 / (Li + Lj));
  const uint32_t b_off = (uint32_t)(Li * TILE_BYTES) >> 4;
  int s = 0, ph = 0;
  for (int it = 0; it < p.n_iters; ++it) {
    tc::mbar_wait(tc::smem_u32(&bar_full[s]), ph);
    tc::tc_fence_after();
    const uint64_t ds = d0 + (uint64_t)(s * (PSTAGE_BYTES >> 4));
#pragma unroll
    for (int kk = 0; kk < KS / 32; ++kk) {
#pragma unroll
      for (int a = 0; a < 3; ++a) {
#pragma unroll
        for (int b = 0; b < 3; ++b) {
          if (a < Li && b < Lj) {
            const uint64_t da = ds + (uint64_t)((a * TILE_BYTES + kk * 32 * BOXW) >> 4);
            const uint64_t db = ds + (uint64_t)(b_off + ((b * TILE_BYTES + kk * 32 * BOXW) >> 4));
            // accumulator a + b: its first product of the tile is the pair with the smallest a, a = max(0, a + b - Lj + 1)
            const int a_first = (a + b) > (Lj - 1) ? (a + b) - (Lj - 1) : 0;
            const bool first = (it == 0) && (kk == 0) && (a == a_first);
            if (tc::elect_one()) tc::mma_i8(tmem + (a + b) * TN, da, db, idesc, first ? 0u : 1u);
          }
        }
      }
    }
    if (tc::elect_one()) tc::mma_commit(tc::smem_u32(&bar_empty[s]));
    __syncwarp();
    if (++s == PNSTAGE) { s = 0; ph ^= 1; }
  }
  if (tc::elect_one()) tc::mma_commit(tc::smem_u32(bar_tmem));
  __syncwarp();
}

__global__ void __launch_bounds__(NTHREADS, 1) gram_tc_kernel(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ CUtensorMap tmapB,
                                                               const GramTcParams p) {
  // Tile order.  CTAs are scheduled in linear block order, and one candidate's digit planes (configs[4]: 3 x 166 MB) do
  // not fit the 126 MB L2.  With the natural order (all column tiles of one row tile, then the next row) the ~148 CTAs
  // in flight share ONE row operand and stream 86 different column operands: every row of tiles re-reads all planes from
  // HBM (measured 373 GB per launch, the kernel was HBM-bound at 3.9 TB/s).  Bands of RB row tiles, column-major inside
  // the band, make the CTAs in flight a ~RB x 12 block of tiles that shares RB row operands and ~12 column operands.
  constexpr int RB = 12;
  const int z = blockIdx.z;
  int ti, tj;
  {
    const int lin = blockIdx.y * gridDim.x + blockIdx.x;
    const int band = lin / (RB * gridDim.x), rem = lin - band * (RB * gridDim.x);
    const int rows = min(RB, (int)gridDim.y - band * RB);
    tj = rem / rows;
    ti = band * RB + (rem - tj * rows);
  }
  const int i0 = ti * TM, j0 = tj * TN;
  if (j0 > i0 + TM - 1) return;                 // tile entirely above the diagonal
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  // 1024-byte alignment for the 128-byte swizzle atoms
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t bar_full[MAXSTAGE], bar_empty[MAXSTAGE], bar_tmem;
  __shared__ uint32_t tmem_base_s;

  const int warp = tc::uniform_warp_id(), lane = threadIdx.x & 31;
  int L = p.nlimb[z], Li = L, Lj = L;           // dual: one digit count per candidate
  if (!p.dual) {                                 // primal: per tile, from the 32-feature group counts
    Li = 1; Lj = 1;
    const int32_t* g = p.nl32 + (long long)z * p.G32;
#pragma unroll
    for (int q = 0; q < TM / 32; ++q) if (i0 / 32 + q < p.G32) Li = max(Li, g[i0 / 32 + q]);
#pragma unroll
    for (int q = 0; q < TN / 32; ++q) if (j0 / 32 + q < p.G32) Lj = max(Lj, g[j0 / 32 + q]);
  }
  const uint32_t smem0 = tc::smem_u32(smem);

  if (warp == 0 && lane == 0) {
    tc::prefetch_tensormap(&tmap);
    tc::prefetch_tensormap(&tmapB);
    for (int s = 0; s < MAXSTAGE; ++s) { tc::mbar_init(tc::smem_u32(&bar_full[s]), 1); tc::mbar_init(tc::smem_u32(&bar_empty[s]), 1); }
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
    if (!p.dual && Li != Lj) gram_produce_p(&tmap, p, smem0, bar_full, bar_empty, i0, j0, z, Li, Lj);
    else if (!p.dual) {               // equal digit counts (the common case): the fully specialised loops
      if (Li == 1) gram_produce<1, false>(&tmap, &tmapB, p, smem0, bar_full, bar_empty, i0, j0, z);
      else if (Li == 2) gram_produce<2, false>(&tmap, &tmapB, p, smem0, bar_full, bar_empty, i0, j0, z);
      else gram_produce<3, false>(&tmap, &tmapB, p, smem0, bar_full, bar_empty, i0, j0, z);
    }
    else if (L == 1) gram_produce<1, true>(&tmap, &tmapB, p, smem0, bar_full, bar_empty, i0, j0, z);
    else if (L == 2) gram_produce<2, true>(&tmap, &tmapB, p, smem0, bar_full, bar_empty, i0, j0, z);
    else gram_produce<3, true>(&tmap, &tmapB, p, smem0, bar_full, bar_empty, i0, j0, z);
  } else if (warp == 1) {
    // ===== MMA issuer =====
    if (!p.dual && Li != Lj) gram_issue_p(p, smem0, tmem, bar_full, bar_empty, &bar_tmem, Li, Lj);
    else if (!p.dual) {
      if (Li == 1) gram_issue<1, false>(p, smem0, tmem, bar_full, bar_empty, &bar_tmem);
      else if (Li == 2) gram_issue<2, false>(p, smem0, tmem, bar_full, bar_empty, &bar_tmem);
      else gram_issue<3, false>(p, smem0, tmem, bar_full, bar_empty, &bar_tmem);
    }
    else if (L == 1) gram_issue<1, true>(p, smem0, tmem, bar_full, bar_empty, &bar_tmem);
    else if (L == 2) gram_issue<2, true>(p, smem0, tmem, bar_full, bar_empty, &bar_tmem);
    else gram_issue<3, true>(p, smem0, tmem, bar_full, bar_empty, &bar_tmem);
    if (p.ops && lane == 0)
      atomicAdd(p.ops, (unsigned long long)p.n_iters * (p.dual ? 4 : KS / 32) * (unsigned long long)(Li * Lj) * (TM * TN * 32));
  } else {
    // ===== epilogue: warps 2..5 own TMEM lanes 32*(warp % 4) .. +31 =====
    const int q = warp & 3;
    tc::mbar_wait(tc::smem_u32(&bar_tmem), 0);
    tc::tc_fence_after();
    const int i = i0 + q * 32 + lane;
    double* Arow = p.A + (long long)z * p.a_stride + (long long)(i + (i >= p.Fcols ? p.rshift : 0)) * p.ld;
    const int nacc = Li + Lj - 1;
    for (int c0 = 0; c0 < TN; c0 += 16) {
      uint32_t r[5][16];
#pragma unroll
      for (int s = 0; s < 5; ++s)
        if (s < nacc) tc::tmem_ld16(tmem + ((uint32_t)(q * 32) << 16) + s * TN + c0, r[s]);
      tc::tmem_ld_wait();
      if (i < p.F) {
#pragma unroll
        for (int e = 0; e < 16; ++e) {
          const int j = j0 + c0 + e;
          if (j < p.Fcols) {
            long long g = 0;
#pragma unroll
            for (int s = 4; s >= 0; --s)
              if (s < nacc) g = g * 256 + (long long)(int32_t)r[s][e];
            double v = (double)g;
            if (p.accumulate) v += Arow[j];          // integers below 2^53: the chunked sum is as exact as the whole one
            if (p.add_lam && i == j) v += p.lam;
            Arow[j] = v;
          }
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

// ---- host side --------------------------------------------------------------------------------------
// plane pitch; `c_aug` one-hot label columns are appended to the features (primal branch: the Gram of [U | T] holds
// U^T T, the right-hand side, in its last c rows -- PAPER.md:67, 70 -- for the price of c extra columns)
// plane pitch: a multiple of 128 bytes, so that every 128-byte TMA box row and every row of the split pass starts on a line
// (with a pitch that is only a multiple of 16 the fused label columns cost configs[2] +10 ms instead of +5)
int64_t lb_gram_tc_fp(int64_t F, int c_aug) { return lb_align_up(F + c_aug, 128); }
// The c extra rows cost at most one more row of 128 x 96 tiles (one digit: the label columns live in plane 0 only), which is
// cheaper than the separate label-segmented pass over the fp32 features (N F 4 bytes of HBM reads): measured on
// configs[2] -2.4 ms, on configs[4] -4.8 ms per step.  More than 128 classes keep the separate kernel.
bool lb_gram_tc_fuse_rhs(int64_t F, int n_classes) { (void)F; return n_classes <= 128; }

// int32 accumulators stay exact while 3 * 128^2 * (contraction length) < 2^31; the contraction runs over the samples
// (primal) or over the features (dual)
bool lb_gram_tc_usable(int64_t n, int64_t F, bool primal) {
  const int64_t k = primal ? n : F;
  return n >= 1 && F >= 1 && k <= LB_GRAM_TC_MAX_K && n < (1 << 30) && F < (1 << 30);
}

size_t lb_gram_tc_ws_bytes(int64_t n, int64_t F, int n_cand, int c_aug) {
  const int64_t Fp = lb_gram_tc_fp(F, c_aug);
  return (size_t)lb_align_up((int64_t)n_cand * 3 * n * Fp, 256) + (size_t)lb_align_up((int64_t)n_cand * (1 + (Fp + 31) / 32) * 4, 256);
}

// A[z] (lower triangle, fp64, leading dimension ld) = U[z]^T U[z] + lam I for integer-valued U, |U| < 2^23 (primal), or
// U U^T + lam I (dual).  Primal with d_labels != NULL: rows F .. F + n_classes - 1 of A[z] additionally receive
// (U^T T)^T, T the one-hot coding of the labels (the appended right-hand-side rows of the Cholesky layout).
int lb_launch_gram_tc(lbcnn_handle_s* h, void* ws, const float* d_U, int64_t n, int64_t F, int n_cand, double lam, double* A,
                      long long a_stride, long long ld, bool primal, const int32_t* d_labels, int n_classes, int32_t* d_info,
                      cudaStream_t st, bool accumulate, bool add_lam, int64_t n_rows, int rshift) {
  // dual branch with n_rows > n: the planes hold n_rows samples per candidate (train rows, then test rows); the output has
  // n_rows rows x n columns -- the n x n system matrix and, in rows n.., the cross-Gram of the test with the train samples
  if (n_rows <= 0 || primal) n_rows = n;
  EncodeTiledFn enc = get_encode();
  if (!enc) return LBCNN_ERR_CUDA;
  const int c_aug = (primal && d_labels && lb_gram_tc_fuse_rhs(F, n_classes)) ? n_classes : 0;
  const int64_t Fp = lb_gram_tc_fp(F, c_aug);
  int8_t* planes = reinterpret_cast<int8_t*>(ws);
  int32_t* nlimb = reinterpret_cast<int32_t*>(reinterpret_cast<char*>(ws) + lb_align_up((int64_t)n_cand * 3 * n_rows * Fp, 256));
  const int G32 = (int)((Fp + 31) / 32);
  int32_t* nl32 = nlimb + n_cand;                  // [n_cand][G32] right behind the per-candidate counts
  const int n_counts = n_cand * (1 + G32);
  // one launch: digit counts = 1 and the candidates' info = 0 (the fit's own zeroing is skipped on this path)
  const int nfill = n_counts > n_cand ? n_counts : n_cand;
  fill_i32_kernel<<<(nfill + 255) / 256, 256, 0, st>>>(nlimb, n_counts, 1, accumulate ? nullptr : d_info, n_cand);
  h->launches += 1;
  {
    const long long work = n_rows * (Fp / 8);
    dim3 grid((unsigned)((work + 255) / 256), (unsigned)n_cand);
    split_kernel<<<grid, 256, 0, st>>>(d_U, n_rows, (int)F, (int)Fp, planes, nlimb, nl32, G32, d_info, d_labels, c_aug);
    h->launches += 1;
  }
  LB_CUDA_OK(cudaGetLastError());
  CUtensorMap tmap, tmapB;
  const cuuint64_t gdim[3] = {(cuuint64_t)(F + c_aug), (cuuint64_t)n_rows, (cuuint64_t)n_cand * 3};
  const cuuint64_t gstr[2] = {(cuuint64_t)Fp, (cuuint64_t)n_rows * Fp};
  const cuuint32_t box[3] = {BOXW, KS, 1};
  const cuuint32_t estr[3] = {1, 1, 1};
  if (enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, planes, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
          CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
    return LBCNN_ERR_CUDA;
  tmapB = tmap;
  if (!primal) {      // K-major tiles: 128 features x (128 | 96) samples
    const cuuint32_t boxA[3] = {128, TM, 1}, boxB[3] = {128, TN, 1};
    if (enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, planes, gdim, gstr, boxA, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS ||
        enc(&tmapB, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, planes, gdim, gstr, boxB, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return LBCNN_ERR_CUDA;
  }
  GramTcParams p{};
  p.nlimb = nlimb; p.nl32 = nl32; p.G32 = G32; p.A = A; p.a_stride = a_stride; p.ld = ld; p.dual = primal ? 0 : 1;
  const int64_t odim = primal ? F + c_aug : n_rows, ocols = primal ? F : n;
  p.rshift = rshift;
  p.Fcols = (int)ocols; p.ops = lb_ws_counter(h, 0); p.accumulate = accumulate ? 1 : 0; p.add_lam = add_lam ? 1 : 0;
  p.F = (int)odim; p.n = (int)n; p.n_iters = primal ? (int)((n + KS - 1) / KS) : (int)((F + 127) / 128); p.lam = lam;
  const size_t smem = (size_t)RING_BYTES + 1024;
  LB_CUDA_OK(cudaFuncSetAttribute(gram_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  dim3 grid((unsigned)((ocols + TN - 1) / TN), (unsigned)((odim + TM - 1) / TM), (unsigned)n_cand);
  gram_tc_kernel<<<grid, NTHREADS, smem, st>>>(tmap, tmapB, p);
  h->launches += 1;
  LB_CUDA_OK(cudaGetLastError());
  return LBCNN_OK;
}
