// score_tc.cu -- K4 on the tensor pipe: logits + argmax + correct count (S1) for integer-valued
// features, as int8 digit products on tcgen05 with int32 TMEM accumulators, the features read ONCE from HBM as fp32.
//
//   logit[n][c] = hs * sum_f u[n][f] w[f][c]
//   u = d0 + 256 d1 + 65536 d2            three balanced radix-256 digits, EXACT for integer |u| <= 8355711; produced in
//                                         shared memory by converter warps from the fp32 tile TMA delivered
//   w[.][c] ~ 2^(e_c - 30) (q0 + 256 q1 + 256^2 q2 + 256^3 q3)   column-scaled, four balanced digits, |error| <= 2^(e_c - 31)
//   sum_f u q = sum_s 256^s T_s,          T_s = sum_{a+b=s} sum_f d_a q_b   (int8 x int8 -> int32, exact for F <= 43690)
// The diagonals s = 2..5 are issued (9 of the 12 digit products, four accumulators of N <= 128 columns = all of TMEM).
// The argmax is taken on these logits; every row carries a RIGOROUS bound E on what was left out (the two dropped
// diagonals and the rounding of w, from the row's digit sums S_a = sum_f |d_a|), and a row whose top-1 / top-2 margin is
// not larger than 2 E -- or that holds a non-integer or out-of-range feature -- is re-evaluated by an exact fp64 kernel.
// The decision therefore equals the fp64 argmax (first index on ties, R12) for every row, at tensor-pipe cost:
// on the configs about one row in a thousand takes the second kernel.
//
// One CTA per (128 test rows, candidate); 10 warps:
//   warp 0      TMA producer: fp32 feature tiles [128 rows][64 features] into a 3-5 stage ring of their own (freed by the
//               converters), the four W digit tiles [N][64 B] into the two-stage digit ring (freed by the MMAs)
//   warp 1      MMA issuer (M = 128, N = 16..128, K = 32; K-major, 64-byte swizzle)
//   warps 2..9  converters: fp32 tile -> three int8 digit tiles in the MMA's swizzled layout (+ digit sums, validity);
//               afterwards warps 2..5 are the epilogue: TMEM -> logits -> argmax / margin test / correct count
#include "internal.h"
#include "tc_common.cuh"
#include <cuda.h>

namespace {

constexpr int NDW = 4;                   // digits of W
constexpr int NDU = 3;                   // digits of U
constexpr int TM = 128;                  // rows per CTA = UMMA M
constexpr int KC = 64;                   // features per stage (64-byte swizzle rows)
constexpr int NTHREADS = 320;
constexpr int NCONV = 256;               // converter threads (warps 2..9)
constexpr uint32_t LAYOUT_SW64 = 4;
constexpr int UF32_BYTES = TM * KC * 4;  // 32 KB fp32 tile (no swizzle: plain [row][64 floats])
constexpr int UD_BYTES = TM * KC;        // 8 KB per U digit tile

struct ScoreTcParams {
  int n, F, c, N;                        // rows, features, classes, padded classes (multiple of 16)
  int n_iters, na, nb, stage_b;           // K steps; fp32 ring stages; digit ring stages and bytes per digit stage
  double hs;
  const double* cscale;                  // [n_cand][N]: 2^(e_c - 30)
  const int32_t* y;
  int32_t* pred; int32_t* correct;
  int32_t* flag_count; int32_t* flag_list;   // rows for the exact kernel: entry = candidate * n + row
};

// ---- W -> column-scaled digit planes ----------------------------------------------------------------------------------
// Wd[cand][4][N][Fp] (class-major rows, feature contiguous = K-major operand), cscale[cand][N] = 2^(e_c - 30) with
// 2^(e_c - 1) <= max_f |w[f][c]| < 2^e_c.  Two passes over W (coalesced, it is F x c floats per candidate):
// column maxima by atomicMax on the bit pattern of |w| (non-negative floats order like their bits), then the digits,
// transposed through shared memory.
constexpr int PF = 64;                   // features per CTA of the two prep kernels

__global__ void __launch_bounds__(256) score_wmax_kernel(const float* __restrict__ W, int F, int c, int N,
                                                         uint32_t* __restrict__ wmax_bits) {
  const int z = blockIdx.y, f0 = blockIdx.x * PF, t = threadIdx.x;
  const float* Wz = W + (long long)z * F * c + (long long)f0 * c;
  const int rows = min(PF, F - f0);
  __shared__ uint32_t s_mx[128];
  for (int cls = t; cls < 128; cls += 256) s_mx[cls] = 0u;
  __syncthreads();
  for (int c0 = 0; c0 < c; c0 += 128) {                      // up to 128 classes per pass
    for (int e = t; e < rows * c; e += 256) {
      const int cls = e % c;
      if (cls >= c0 && cls < c0 + 128) {
        const uint32_t b = __float_as_uint(fabsf(Wz[e]));
        if (b > s_mx[cls - c0]) atomicMax(&s_mx[cls - c0], b);
      }
    }
    __syncthreads();
    for (int cls = t; cls < 128 && c0 + cls < c; cls += 256) {
      if (s_mx[cls]) atomicMax(&wmax_bits[(long long)z * N + c0 + cls], s_mx[cls]);
      s_mx[cls] = 0u;
    }
    __syncthreads();
  }
}

__global__ void __launch_bounds__(256) score_quant_kernel(const float* __restrict__ W, int F, int c, int N, int Fp,
                                                          const uint32_t* __restrict__ wmax_bits, int8_t* __restrict__ Wd,
                                                          double* __restrict__ cscale) {
  extern __shared__ int32_t sq[];                             // [PF][c + 1] quantised values of this feature tile
  const int z = blockIdx.y, f0 = blockIdx.x * PF, t = threadIdx.x;
  const float* Wz = W + (long long)z * F * c + (long long)f0 * c;
  const int rows = min(PF, F - f0), pitch = c + 1;
  for (int e = t; e < PF * c; e += 256) {
    const int r = e / c, cls = e - r * c;
    int v = 0;
    if (r < rows) {
      const float mx = __uint_as_float(wmax_bits[(long long)z * N + cls]);
      int ex = 0;
      if (mx > 0.0f && mx < 3.0e38f) frexpf(mx, &ex);         // mx = m 2^ex, m in [0.5, 1)
      v = __double2int_rn((double)Wz[e] * scalbn(1.0, 30 - ex));
    }
    sq[r * pitch + cls] = v;
  }
  if (blockIdx.x == 0)
    for (int cls = t; cls < N; cls += 256) {
      int ex = 0;
      if (cls < c) {
        const float mx = __uint_as_float(wmax_bits[(long long)z * N + cls]);
        if (mx > 0.0f && mx < 3.0e38f) frexpf(mx, &ex);
      }
      cscale[(long long)z * N + cls] = scalbn(1.0, ex - 30);
    }
  __syncthreads();
  // thread -> (class, four consecutive features): one 32-bit store per digit plane, 64 contiguous bytes per class row
  const long long plane = (long long)N * Fp;
  for (int e = t; e < N * (PF / 4); e += 256) {
    const int cls = e / (PF / 4), g = (e - cls * (PF / 4)) * 4;
    if (f0 + g >= Fp) continue;
    uint32_t w[NDW] = {0u, 0u, 0u, 0u};
    if (cls < c) {
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        int v = sq[(g + q) * pitch + cls];
#pragma unroll
        for (int a = 0; a < NDW; ++a) {
          const int d = (int)(int8_t)(v & 0xFF);
          w[a] |= (uint32_t)(d & 0xFF) << (8 * q);
          v = (v - d) >> 8;
        }
      }
    }
    int8_t* dst = Wd + ((long long)z * NDW * N + cls) * Fp + f0 + g;
#pragma unroll
    for (int a = 0; a < NDW; ++a) *reinterpret_cast<uint32_t*>(dst + a * plane) = w[a];
  }
}

// int8 output layer q[F][c] -> the single digit plane Wd[cand][N][Fp] (class-major), cscale = 1
__global__ void __launch_bounds__(256) score_q8_prep_kernel(const int8_t* __restrict__ Wq, int F, int c, int N, int Fp,
                                                            int8_t* __restrict__ Wd, double* __restrict__ cscale) {
  extern __shared__ int8_t sq8[];                             // [PF][c + 1]
  const int z = blockIdx.y, f0 = blockIdx.x * PF, t = threadIdx.x;
  const int8_t* Wz = Wq + (long long)z * F * c + (long long)f0 * c;
  const int rows = min(PF, F - f0), pitch = c + 1;
  for (int e = t; e < PF * c; e += 256) {
    const int r = e / c, cls = e - r * c;
    sq8[r * pitch + cls] = (r < rows) ? Wz[e] : (int8_t)0;
  }
  if (blockIdx.x == 0)
    for (int cls = t; cls < N; cls += 256) cscale[(long long)z * N + cls] = 1.0;
  __syncthreads();
  for (int e = t; e < N * (PF / 4); e += 256) {
    const int cls = e / (PF / 4), g = (e - cls * (PF / 4)) * 4;
    uint32_t w = 0u;
    if (cls < c) {
#pragma unroll
      for (int q = 0; q < 4; ++q) w |= (uint32_t)(uint8_t)sq8[(g + q) * pitch + cls] << (8 * q);
    }
    *reinterpret_cast<uint32_t*>(Wd + ((long long)z * N + cls) * Fp + f0 + g) = w;
  }
}

// ---- the scoring kernel -----------------------------------------------------------------------------------------------
constexpr int MAXA = 6, MAXB = 2;        // fp32 feature ring (32 KB per stage) / digit ring (U digits + W digits)

// NW digit planes of W, diagonals SMIN .. NDU + NW - 2 issued: <4, 2> = fp32 W as four column-scaled digits (nine of the
// twelve products, error-bounded); <1, 0> = an int8 output layer (lbcnn_elm_score_q): all three products, EXACT integer logits
template <int NW, int SMIN>
__global__ void __launch_bounds__(NTHREADS, 1) score_tc_kernel(const __grid_constant__ CUtensorMap tmapU,
                                                               const __grid_constant__ CUtensorMap tmapW, const ScoreTcParams p) {
  constexpr int NACC = NDU + NW - 1 - SMIN;      // accumulators (diagonals kept)
  const int z = blockIdx.y;
  const int i0 = blockIdx.x * TM;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t bar_fullA[MAXA], bar_emptyA[MAXA], bar_fullW[MAXB], bar_conv[MAXB], bar_emptyB[MAXB], bar_tmem;
  __shared__ uint32_t tmem_base_s;
  __shared__ int32_t row_s[TM][4];               // digit sums S0, S1, S2 and the invalid-feature flag of every row
  const int warp = tc::uniform_warp_id(), lane = threadIdx.x & 31;
  const uint32_t smem0 = tc::smem_u32(smem);
  const int N = p.N, na = p.na, nb = p.nb, stage_b = p.stage_b;
  const int w_tile = N * KC;                     // bytes of one W digit tile
  const int off_b = na * UF32_BYTES;             // the digit ring starts behind the fp32 ring
  const int off_w = NDU * UD_BYTES;              // W digit tiles inside a digit stage (behind the three U digit tiles)

  if (warp == 0 && lane == 0) {
    tc::prefetch_tensormap(&tmapU);
    tc::prefetch_tensormap(&tmapW);
    for (int s = 0; s < MAXA; ++s) {
      tc::mbar_init(tc::smem_u32(&bar_fullA[s]), 1);
      tc::mbar_init(tc::smem_u32(&bar_emptyA[s]), NCONV / 32);
    }
    for (int s = 0; s < MAXB; ++s) {
      tc::mbar_init(tc::smem_u32(&bar_fullW[s]), 1);
      tc::mbar_init(tc::smem_u32(&bar_conv[s]), NCONV / 32);
      tc::mbar_init(tc::smem_u32(&bar_emptyB[s]), 1);
    }
    tc::mbar_init(tc::smem_u32(&bar_tmem), 1);
    tc::fence_barrier_init();
  }
  if (warp == 1) tc::tmem_alloc(tc::smem_u32(&tmem_base_s), 512);
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t tmem = tmem_base_s;

  if (warp == 0) {
    // ===== TMA producer: two independent streams -- fp32 feature tiles into ring A (freed by the converters), W digit tiles
    // into ring B (freed by the MMAs).  Whichever slot is free is filled, so up to `na` feature tiles are in flight. =====
    int ia = 0, sa = 0, pa = 0, ib = 0, sb = 0, pb = 0;
    const int n = p.n_iters;
    while (ia < n || ib < n) {
      if (ia < n && tc::mbar_try_wait(tc::smem_u32(&bar_emptyA[sa]), pa ^ 1)) {
        if (tc::elect_one()) {
          const uint32_t full = tc::smem_u32(&bar_fullA[sa]);
          tc::mbar_arrive_expect_tx(full, UF32_BYTES);
          tc::tma_load_3d(smem0 + sa * UF32_BYTES, &tmapU, full, ia * KC, i0, z);
        }
        __syncwarp();
        ++ia;
        if (++sa == na) { sa = 0; pa ^= 1; }
      }
      if (ib < n && tc::mbar_try_wait(tc::smem_u32(&bar_emptyB[sb]), pb ^ 1)) {
        if (tc::elect_one()) {
          const uint32_t full = tc::smem_u32(&bar_fullW[sb]);
          tc::mbar_arrive_expect_tx(full, (uint32_t)(NW * w_tile));
          const uint32_t base = smem0 + off_b + sb * stage_b + off_w;
#pragma unroll
          for (int b = 0; b < NW; ++b) tc::tma_load_3d(base + b * w_tile, &tmapW, full, ib * KC, 0, z * NW + b);
        }
        __syncwarp();
        ++ib;
        if (++sb == nb) { sb = 0; pb ^= 1; }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer: diagonals s = a + b = SMIN .. into accumulators 0 .. NACC-1 =====
    const uint32_t idesc = tc::idesc_i8(TM, N, 1, 1, 0, 0);
    const uint64_t d0 = tc::smem_desc(smem0, 16, 8 * KC, LAYOUT_SW64);
    int s = 0, ph = 0;
    for (int it = 0; it < p.n_iters; ++it) {
      tc::mbar_wait(tc::smem_u32(&bar_fullW[s]), ph);     // W digit tiles have landed
      tc::mbar_wait(tc::smem_u32(&bar_conv[s]), ph);      // U digit tiles are written
      tc::tc_fence_after();
      const uint64_t ds = d0 + (uint64_t)((off_b + s * stage_b) >> 4);
#pragma unroll
      for (int kk = 0; kk < KC / 32; ++kk) {
#pragma unroll
        for (int sd = SMIN; sd <= NDU + NW - 2; ++sd) {
#pragma unroll
          for (int a = 0; a < NDU; ++a) {
            const int b = sd - a;
            if (b >= 0 && b < NW) {
              const uint64_t da = ds + (uint64_t)((a * UD_BYTES + kk * 32) >> 4);
              const uint64_t db = ds + (uint64_t)((off_w + b * w_tile + kk * 32) >> 4);
              const int a_first = (sd - (NW - 1)) > 0 ? sd - (NW - 1) : 0;             // smallest a of this diagonal
              const bool first = (kk == 0) && (a == a_first);
              if (tc::elect_one()) tc::mma_i8(tmem + (sd - SMIN) * N, da, db, idesc, (first && it == 0) ? 0u : 1u);
            }
          }
        }
      }
      if (tc::elect_one()) tc::mma_commit(tc::smem_u32(&bar_emptyB[s]));
      __syncwarp();
      if (++s == nb) { s = 0; ph ^= 1; }
    }
    if (tc::elect_one()) tc::mma_commit(tc::smem_u32(&bar_tmem));
    __syncwarp();
  } else {
    // ===== converters: fp32 tile -> three swizzled int8 digit tiles =====
    // thread tc owns the 16-byte chunk column cc = tc % 16 (features 4 cc .. 4 cc + 3) of rows tc / 16 + 16 m, m = 0..7
    const int tcid = threadIdx.x - 64, cc = tcid & 15, r_base = tcid >> 4;
    int S0[8], S1[8], S2[8];
    uint32_t bad = 0;
#pragma unroll
    for (int m = 0; m < 8; ++m) { S0[m] = 0; S1[m] = 0; S2[m] = 0; }
    int sa = 0, pa = 0, sb = 0, pb = 0;
    for (int it = 0; it < p.n_iters; ++it) {
      tc::mbar_wait(tc::smem_u32(&bar_fullA[sa]), pa);          // the fp32 tile has landed
      tc::mbar_wait(tc::smem_u32(&bar_emptyB[sb]), pb ^ 1);     // the digit stage is free (its MMAs of two steps ago are done)
      const uint8_t* st = smem + sa * UF32_BYTES;
      uint8_t* sd = smem + off_b + sb * stage_b;
#pragma unroll
      for (int m = 0; m < 8; ++m) {
        const int r = r_base + 16 * m;
        const float4 x = *reinterpret_cast<const float4*>(st + r * (KC * 4) + cc * 16);
        const int v0 = (int)x.x, v1 = (int)x.y, v2 = (int)x.z, v3 = (int)x.w;
        const bool ok = ((float)v0 == x.x) && ((float)v1 == x.y) && ((float)v2 == x.z) && ((float)v3 == x.w);
        const uint32_t a0 = (uint32_t)(v0 + 128), a1 = (uint32_t)(v1 + 128), a2 = (uint32_t)(v2 + 128), a3 = (uint32_t)(v3 + 128);
        const uint32_t b0 = (uint32_t)(v0 + 32896), b1 = (uint32_t)(v1 + 32896), b2 = (uint32_t)(v2 + 32896), b3 = (uint32_t)(v3 + 32896);
        const bool range = ((b0 + 0x800000u) | (b1 + 0x800000u) | (b2 + 0x800000u) | (b3 + 0x800000u)) < 0x1000000u;
        if (!(ok && range)) bad |= 1u << m;
        // byte `sel` of four words -> one word
        const uint32_t w0 = __byte_perm(__byte_perm((uint32_t)v0, (uint32_t)v1, 0x0040), __byte_perm((uint32_t)v2, (uint32_t)v3, 0x0040), 0x5410);
        const uint32_t w1 = __byte_perm(__byte_perm(a0, a1, 0x0051), __byte_perm(a2, a3, 0x0051), 0x5410);
        const uint32_t w2 = __byte_perm(__byte_perm(b0, b1, 0x0062), __byte_perm(b2, b3, 0x0062), 0x5410);
        S0[m] += (int)__vsads4(w0, 0u); S1[m] += (int)__vsads4(w1, 0u); S2[m] += (int)__vsads4(w2, 0u);
        // 64-byte swizzle: 16-byte chunk index (cc / 4) XOR bits 1..2 of the row; word cc % 4 inside the chunk
        const uint32_t off = (uint32_t)r * KC + ((((uint32_t)cc >> 2) ^ (((uint32_t)r >> 1) & 3u)) << 4) + (((uint32_t)cc & 3u) << 2);
        uint8_t* ud = sd + off;
        *reinterpret_cast<uint32_t*>(ud) = w0;
        *reinterpret_cast<uint32_t*>(ud + UD_BYTES) = w1;
        *reinterpret_cast<uint32_t*>(ud + 2 * UD_BYTES) = w2;
      }
      tc::fence_proxy_async();                 // generic-proxy writes of the digit tiles -> visible to the MMA's async proxy
      __syncwarp();
      if (lane == 0) {
        tc::mbar_arrive(tc::smem_u32(&bar_conv[sb]));           // digits ready for the MMAs
        tc::mbar_arrive(tc::smem_u32(&bar_emptyA[sa]));         // fp32 slot free for the next TMA
      }
      if (++sa == na) { sa = 0; pa ^= 1; }
      if (++sb == nb) { sb = 0; pb ^= 1; }
    }
    // digit sums of every row: reduce over the 16 threads (a half warp) that share the row
#pragma unroll
    for (int m = 0; m < 8; ++m) {
      int s0 = S0[m], s1 = S1[m], s2 = S2[m], bd = (int)((bad >> m) & 1u);
#pragma unroll
      for (int d = 8; d >= 1; d >>= 1) {
        s0 += __shfl_xor_sync(0xffffffffu, s0, d); s1 += __shfl_xor_sync(0xffffffffu, s1, d);
        s2 += __shfl_xor_sync(0xffffffffu, s2, d); bd |= __shfl_xor_sync(0xffffffffu, bd, d);
      }
      if (cc == 0) { const int r = r_base + 16 * m; row_s[r][0] = s0; row_s[r][1] = s1; row_s[r][2] = s2; row_s[r][3] = bd; }
    }
    asm volatile("bar.sync 1, 256;" ::: "memory");
    if (warp < 6) {
      // ===== epilogue (warps 2..5): TMEM lanes 32 (warp % 4) .. +31 =====
      const int q = warp & 3, r = q * 32 + lane;
      const long long row = (long long)i0 + r;
      tc::mbar_wait(tc::smem_u32(&bar_tmem), 0);
      tc::tc_fence_after();
      const double* cs = p.cscale + (long long)z * N;
      double best = 0.0, second = 0.0, cs_max = 0.0;
      int bidx = -1, have2 = 0;
      for (int c0 = 0; c0 < N; c0 += 16) {
        uint32_t acc[NACC][16];
#pragma unroll
        for (int sd = 0; sd < NACC; ++sd) tc::tmem_ld16(tmem + ((uint32_t)(q * 32) << 16) + sd * N + c0, acc[sd]);
        tc::tmem_ld_wait();
#pragma unroll
        for (int e = 0; e < 16; ++e) {
          const int j = c0 + e;
          if (j < p.c) {
            long long g = 0;
#pragma unroll
            for (int sd = NACC - 1; sd >= 0; --sd) g = g * 256 + (long long)(int32_t)acc[sd][e];
            const double csj = cs[j];
            const double l = (double)g * csj;
            cs_max = fmax(cs_max, csj);
            if (bidx < 0) { best = l; bidx = j; }
            else if (l > best) { second = best; have2 = 1; best = l; bidx = j; }        // strict: the first maximum stays
            else if (!have2 || l > second) { second = l; have2 = 1; }
          }
        }
      }
      tc::tc_fence_before();
      int ok = 0;
      if (row < p.n) {
        // what the issued diagonals leave out, in the units of l (= true logit / (65536 hs)): the dropped diagonals 0 and 1
        // (|d q| <= 128 |d|) and the rounding of w (half a unit of its last digit per feature)
        const double s0 = (double)row_s[r][0], s1 = (double)row_s[r][1], s2 = (double)row_s[r][2];
        const double E = (SMIN == 0) ? 0.0 :       // all diagonals and integer weights: the logits are exact, only ties go on
            cs_max * ((128.0 * 257.0 * s0 + 32768.0 * s1) + 0.5 * (s0 + 256.0 * s1 + 65536.0 * s2)) * (1.0 / 65536.0);
        const bool exact = row_s[r][3] != 0 || !(best - second > 2.0 * E);
        if (exact) {
          const int slot = atomicAdd(p.flag_count, 1);
          p.flag_list[slot] = (int32_t)((long long)z * p.n + row);
        } else {
          if (p.pred) p.pred[(long long)z * p.n + row] = bidx;
          if (p.y && p.y[row] == bidx) ok = 1;
        }
      }
      ok = __reduce_add_sync(0xffffffffu, ok);
      if (lane == 0 && ok && p.correct) atomicAdd(&p.correct[z], ok);
    }
  }
  __syncthreads();
  if (warp == 1) { tc::tc_fence_after(); tc::tmem_dealloc(tmem, 512); }
}

// ---- exact re-evaluation of the flagged rows (fp64) ---------------------------------------------------------------------
// One CTA per flagged row, the 128 threads split the FEATURES (thread t takes f = t, t + 128, ...: coalesced reads of the
// row, eight classes at a time in registers), then a fixed-order tree over the threads: deterministic, every product
// exact in fp64 (fp32 x fp32), only the order of the fp64 additions differs from the oracle's plain loop.
template <typename TW>
__global__ void __launch_bounds__(128) score_exact_kernel(const float* __restrict__ U, long long n, long long F,
                                                          const TW* __restrict__ W, int c, const int32_t* __restrict__ y,
                                                          const int32_t* __restrict__ flag_count, const int32_t* __restrict__ flag_list,
                                                          int32_t* __restrict__ pred, int32_t* __restrict__ correct) {
  __shared__ double red[4][8];
  const int t = threadIdx.x, lane = t & 31, wp = t >> 5, total = *flag_count;
  for (int idx = blockIdx.x; idx < total; idx += gridDim.x) {
    const long long e = flag_list[idx];
    const long long z = e / n, row = e - z * n;
    const float* Ur = U + (z * n + row) * F;
    const TW* Wz = W + z * F * c;
    double bestv = 0.0; int besti = -1;
    for (int c0 = 0; c0 < c; c0 += 8) {
      double acc[8];
#pragma unroll
      for (int q = 0; q < 8; ++q) acc[q] = 0.0;
      const int nc = (c - c0 < 8) ? c - c0 : 8;
      for (long long f = t; f < F; f += 128) {
        const double u = (double)Ur[f];
        const TW* wr = Wz + f * c + c0;
#pragma unroll
        for (int q = 0; q < 8; ++q)
          if (q < nc) acc[q] = fma(u, (double)wr[q], acc[q]);
      }
#pragma unroll
      for (int q = 0; q < 8; ++q) {
#pragma unroll
        for (int d = 16; d >= 1; d >>= 1) acc[q] += __shfl_xor_sync(0xffffffffu, acc[q], d);
      }
      __syncthreads();
      if (lane == 0) {
#pragma unroll
        for (int q = 0; q < 8; ++q) red[wp][q] = acc[q];
      }
      __syncthreads();
      if (t == 0) {
        for (int q = 0; q < nc; ++q) {
          const double l = (red[0][q] + red[1][q]) + (red[2][q] + red[3][q]);
          if (besti < 0 || l > bestv) { bestv = l; besti = c0 + q; }                 // first index on ties
        }
      }
    }
    if (t == 0) {
      if (pred) pred[z * n + row] = besti;
      if (y && correct && y[row] == besti) atomicAdd(&correct[z], 1);
    }
  }
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

// ---- host side ----------------------------------------------------------------------------------------------------------
namespace {
struct ScoreTcLayout { size_t wd, cscale, zero0, wmax, flag_count, flag_list, total; size_t zero_bytes; int N; int64_t Fp; };
void score_tc_layout(int64_t n, int64_t F, int c, int n_cand, ScoreTcLayout* L) {
  L->N = (c + 15) / 16 * 16;
  L->Fp = lb_align_up(F, KC);
  size_t off = 0;
  L->wd = off;         off += (size_t)lb_align_up((int64_t)n_cand * NDW * L->N * L->Fp, 256);
  L->cscale = off;     off += (size_t)lb_align_up((int64_t)n_cand * L->N * 8, 256);
  L->zero0 = off;                                   // [wmax bits | flag counter]: cleared by one cudaMemsetAsync per call
  L->wmax = off;       off += (size_t)lb_align_up((int64_t)n_cand * L->N * 4, 256);
  L->flag_count = off; off += 256;
  L->zero_bytes = off - L->zero0;
  L->flag_list = off;  off += (size_t)lb_align_up((int64_t)n_cand * n * 4, 256);
  L->total = off;
}
}  // namespace

// the tensor-core scorer takes integer-valued features with up to 128 classes; everything else stays on the fp64 kernel
bool lb_score_tc_worthwhile(int64_t n, int64_t F, int n_classes, int n_cand) {
  // below ~1e9 multiply-adds the two preparation kernels and the second pass cost more than the fp64 kernel's whole run
  return (double)n * (double)F * (double)n_classes * (double)n_cand >= 1.0e9;
}

bool lb_score_tc_usable(const float* d_H, int64_t n, int64_t F, int n_classes, int n_cand) {
  return n_classes <= 128 && (F % 4) == 0 && F <= 43690 && F >= 4 && (reinterpret_cast<uintptr_t>(d_H) % 16) == 0 &&
         (int64_t)n_cand * n < (1LL << 31) && n < (1 << 30) && n_cand <= 65535;
}

size_t lb_score_tc_ws_bytes(int64_t n, int64_t F, int n_classes, int n_cand) {
  ScoreTcLayout L;
  score_tc_layout(n, F, n_classes, n_cand, &L);
  return L.total;
}

namespace {
// d_Wq != NULL: int8 output layer (one digit plane, exact integer logits); else fp32 d_W as four column-scaled digit planes
int launch_score_common(lbcnn_handle_s* h, void* ws, const float* d_H, int64_t n, int64_t F, float h_scale, const float* d_W,
                        const int8_t* d_Wq, int n_classes, const int32_t* d_labels, int n_cand, int32_t* d_pred,
                        int32_t* d_correct, cudaStream_t st, bool keep_correct) {
  EncodeTiledFn enc = get_encode();
  if (!enc) return LBCNN_ERR_CUDA;
  LbPhase ph(h, LBCNN_PHASE_SCORE, st);
  ScoreTcLayout L;
  score_tc_layout(n, F, n_classes, n_cand, &L);
  char* base = reinterpret_cast<char*>(ws);
  int8_t* Wd = reinterpret_cast<int8_t*>(base + L.wd);
  double* cscale = reinterpret_cast<double*>(base + L.cscale);
  uint32_t* wmax = reinterpret_cast<uint32_t*>(base + L.wmax);
  int32_t* flag_count = reinterpret_cast<int32_t*>(base + L.flag_count);
  int32_t* flag_list = reinterpret_cast<int32_t*>(base + L.flag_list);
  const int N = L.N, c = n_classes, NW = d_Wq ? 1 : NDW;
  const int Fp = (int)L.Fp;
  LB_CUDA_OK(cudaMemsetAsync(base + L.zero0, 0, L.zero_bytes, st));
  if (d_correct && !keep_correct) LB_CUDA_OK(cudaMemsetAsync(d_correct, 0, (size_t)n_cand * 4, st));
  {
    dim3 grid((unsigned)(Fp / PF), (unsigned)n_cand);
    if (d_Wq) {
      score_q8_prep_kernel<<<grid, 256, (size_t)PF * (c + 1), st>>>(d_Wq, (int)F, c, N, Fp, Wd, cscale);
      h->launches += 1;
    } else {
      score_wmax_kernel<<<grid, 256, 0, st>>>(d_W, (int)F, c, N, wmax);
      const size_t sm = (size_t)PF * (c + 1) * 4;
      score_quant_kernel<<<grid, 256, sm, st>>>(d_W, (int)F, c, N, Fp, wmax, Wd, cscale);
      h->launches += 2;
    }
    LB_CUDA_OK(cudaGetLastError());
  }
  CUtensorMap tmapU, tmapW;
  {
    const cuuint64_t gdim[3] = {(cuuint64_t)F, (cuuint64_t)n, (cuuint64_t)n_cand};
    const cuuint64_t gstr[2] = {(cuuint64_t)F * 4, (cuuint64_t)n * F * 4};
    const cuuint32_t box[3] = {KC, TM, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    if (enc(&tmapU, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(d_H), gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return LBCNN_ERR_CUDA;
  }
  {
    const cuuint64_t gdim[3] = {(cuuint64_t)Fp, (cuuint64_t)N, (cuuint64_t)n_cand * NW};
    const cuuint64_t gstr[2] = {(cuuint64_t)Fp, (cuuint64_t)N * Fp};
    const cuuint32_t box[3] = {KC, (cuuint32_t)N, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    if (enc(&tmapW, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, Wd, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return LBCNN_ERR_CUDA;
  }
  ScoreTcParams p{};
  p.n = (int)n; p.F = (int)F; p.c = c; p.N = N; p.n_iters = Fp / KC; p.hs = (double)h_scale;
  // shared memory: two digit stages (U digits + W digits) and as many 32 KB fp32 feature stages as fit beside them
  p.stage_b = NDU * UD_BYTES + NW * N * KC;
  p.nb = MAXB;
  p.na = (int)(((size_t)h->max_smem_optin - 4096 - (size_t)p.nb * p.stage_b) / (size_t)UF32_BYTES);
  if (p.na > MAXA) p.na = MAXA;
  if (p.na < 2) return LBCNN_ERR_INVALID_ARG;
  p.cscale = cscale; p.y = d_labels; p.pred = d_pred; p.correct = d_correct; p.flag_count = flag_count; p.flag_list = flag_list;
  const size_t smem = (size_t)p.na * UF32_BYTES + (size_t)p.nb * p.stage_b + 1024;
  dim3 grid((unsigned)((n + TM - 1) / TM), (unsigned)n_cand);
  if (d_Wq) {
    LB_CUDA_OK(cudaFuncSetAttribute(score_tc_kernel<1, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    score_tc_kernel<1, 0><<<grid, NTHREADS, smem, st>>>(tmapU, tmapW, p);
    score_exact_kernel<int8_t><<<2 * h->n_sm, 128, 0, st>>>(d_H, n, F, d_Wq, c, d_labels, flag_count, flag_list, d_pred, d_correct);
  } else {
    LB_CUDA_OK(cudaFuncSetAttribute(score_tc_kernel<NDW, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    score_tc_kernel<NDW, 2><<<grid, NTHREADS, smem, st>>>(tmapU, tmapW, p);
    score_exact_kernel<float><<<2 * h->n_sm, 128, 0, st>>>(d_H, n, F, d_W, c, d_labels, flag_count, flag_list, d_pred, d_correct);
  }
  h->launches += 2;
  LB_CUDA_OK(cudaGetLastError());
  return LBCNN_OK;
}
}  // namespace

int lb_launch_score_tc(lbcnn_handle_s* h, void* ws, const float* d_H, int64_t n, int64_t F, float h_scale, const float* d_W,
                       int n_classes, const int32_t* d_labels, int n_cand, int32_t* d_pred, int32_t* d_correct,
                       cudaStream_t st, bool keep_correct) {
  return launch_score_common(h, ws, d_H, n, F, h_scale, d_W, nullptr, n_classes, d_labels, n_cand, d_pred, d_correct, st, keep_correct);
}

// S1 with an int8 output layer ("weights represented as 8 bits integers"): exact integer logits
int lb_launch_score_q8(lbcnn_handle_s* h, void* ws, const float* d_H, int64_t n, int64_t F, const int8_t* d_Wq, int n_classes,
                       const int32_t* d_labels, int n_cand, int32_t* d_pred, int32_t* d_correct, cudaStream_t st) {
  return launch_score_common(h, ws, d_H, n, F, 1.0f, nullptr, d_Wq, n_classes, d_labels, n_cand, d_pred, d_correct, st, false);
}

// ---- <= 8-bit fixed-point output layer (PAPER.md:94, 98 Cell 12, 131; R16) ------------------------------------------
namespace {
__global__ void __launch_bounds__(256) wq_max_kernel(const float* __restrict__ W, long long per_cand, uint32_t* __restrict__ mx_bits) {
  const long long z = blockIdx.y;
  const float* Wz = W + z * per_cand;
  uint32_t m = 0u;
  for (long long e = (long long)blockIdx.x * 256 + threadIdx.x; e < per_cand; e += (long long)gridDim.x * 256)
    m = max(m, __float_as_uint(fabsf(Wz[e])));
  m = __reduce_max_sync(0xffffffffu, m);
  if ((threadIdx.x & 31) == 0 && m) atomicMax(&mx_bits[z], m);
}
// q = clip(rint(w * (qmax / max|W|)), -qmax, qmax): the product in fp64, round half to even -- the oracle does the same
__global__ void __launch_bounds__(256) wq_quant_kernel(const float* __restrict__ W, long long per_cand, const uint32_t* __restrict__ mx_bits,
                                                       int qmax, int8_t* __restrict__ Wq) {
  const long long z = blockIdx.y;
  const float m = __uint_as_float(mx_bits[z]);
  const double sf = (m > 0.0f) ? (double)qmax / (double)m : 0.0;
  for (long long e = (long long)blockIdx.x * 256 + threadIdx.x; e < per_cand; e += (long long)gridDim.x * 256) {
    int q = __double2int_rn((double)W[z * per_cand + e] * sf);
    q = max(-qmax, min(qmax, q));
    Wq[z * per_cand + e] = (int8_t)q;
  }
}
// scale[z] = max|W| / qmax (fp32, one rounding of the fp64 quotient), in place over the bit pattern of the maximum
__global__ void wq_scale_kernel(uint32_t* __restrict__ mx_bits, int n_cand, int qmax) {
  const int z = blockIdx.x * blockDim.x + threadIdx.x;
  if (z < n_cand) {
    const float m = __uint_as_float(mx_bits[z]);
    reinterpret_cast<float*>(mx_bits)[z] = (float)((double)m / (double)qmax);
  }
}
}  // namespace

int lb_launch_quantize_w(lbcnn_handle_s* h, const float* d_W, int64_t F, int n_classes, int n_cand, int bits, int8_t* d_Wq,
                         float* d_scale, cudaStream_t st) {
  const int qmax = (1 << (bits - 1)) - 1;
  const long long per = (long long)F * n_classes;
  uint32_t* mx = reinterpret_cast<uint32_t*>(d_scale);
  LB_CUDA_OK(cudaMemsetAsync(mx, 0, (size_t)n_cand * 4, st));
  const unsigned gx = (unsigned)((per + 256 * 8 - 1) / (256 * 8) < 1 ? 1 : ((per + 256 * 8 - 1) / (256 * 8) > 1024 ? 1024 : (per + 256 * 8 - 1) / (256 * 8)));
  dim3 grid(gx, (unsigned)n_cand);
  wq_max_kernel<<<grid, 256, 0, st>>>(d_W, per, mx);
  wq_quant_kernel<<<grid, 256, 0, st>>>(d_W, per, mx, qmax, d_Wq);
  wq_scale_kernel<<<(n_cand + 255) / 256, 256, 0, st>>>(mx, n_cand, qmax);
  h->launches += 3;
  LB_CUDA_OK(cudaGetLastError());
  return LBCNN_OK;
}
