// expand_tc.cu -- K1 on the tensor pipe: the LB-CNN expander for FULL convolutions with
// non-overlapping pooling, as exact integer implicit GEMMs on tcgen05.mma kind::i8 (int32 accumulators in TMEM).
//
// Layer 1 ("patch GEMM").  A pooled output position (i,j) sees a (P+k-1)^2 x Cin patch of uint8 pixels; all P*P
// conv outputs under its pooling window are linear in that one patch.  A1 = [pooled position][patch bytes]
// (built ONCE per CTA in shared memory, shared by every candidate), B1 = [patch byte][o * P*P + phase] holds the
// candidate's +-1 taps shifted per pool phase (zero elsewhere): one u8 x s8 -> s32 MMA chain per 128 positions
// gives every pre-pool value of the tile, the pool is a max over P*P adjacent TMEM columns of the thread's own
// lane -- no shuffles ("Nonlinearity achieved in Max-pool").
// Layer 2 ("tap-shifted implicit GEMM").  The pooled layer-1 map (|v| < 8192) is written to shared memory as
// two int8 digits v = 64 hi + lo (lo = v & 63, hi = v >> 6), split into P2*P2 phase planes
// plane[sy][sx](i,j) = a[P2 i + sy][P2 j + sx] that share one zero halo.  For output phase (py,px) and tap
// (dy,dx) the A operand is a plane shifted by a constant number of positions = a different start address of a
// K-major no-swizzle descriptor; the k*k taps accumulate into one TMEM accumulator, the B operand holds +-1
// (lo digits) and +-64 (hi digits), so the int32 result is the exact convolution.  Pool = max over the phase
// accumulators; flatten C,H,W; one multiply by feature_scale; H written once.
//
// One CTA = a batch of B images x a range of candidates, 19 warps, warp specialised, everything handed over
// through mbarriers so that the tensor pipe, the TMEM reads and the ALU epilogues of neighbouring candidates overlap:
//   warp 0       layer-1 MMA issuer (+ bulk-copy of the candidate's prepared B1)   -> accumulator ring R1 (4 slots)
//   warps 1, 18  layer-2 MMA issuers, one pool row each (warp 1 also bulk-copies B2); they wait for the planes
//                                                                                  -> accumulator ring R2 (2 slots)
//   warps 2-9    E1: R1 -> max-pool -> digits -> phase planes (double buffered)  [single layer: -> H, warps 2-17]
//   warps 10-17  E2: R2 -> max-pool -> scale -> H
// With 2x2 pooling the two px phases of a pool row read the same shifted plane, so one N = 2 N2 MMA feeds both.
// The +-1 kernel sets are re-laid-out once per launch by a small kernel into the exact shared-memory images of
// B1 / B2 (handle-owned scratch), so the hot loop stages them with one cp.async.bulk each.
// Measured on B200: an MMA with M = 128 reads (128 + N) x 32 operand bytes from shared memory at 128 B/clk, so
// these small-N MMAs are bound by shared-memory bandwidth (32 + N/4 clk), not by the tensor pipe (N/2 clk).
// Anything outside this kernel's envelope (depthwise, overlapping / padded / cover_all pooling, bias, three
// layers, wide layers) takes the exact SIMT kernel in expand.cu.
#include "internal.h"
#include "tc_common.cuh"

namespace {

constexpr int XT_WARPS = 19;
constexpr int XT_THREADS = XT_WARPS * 32;

struct XtcParams {
  const uint8_t* img; long long n_img; int H, W, C;
  long long out_rows;            // rows per candidate of the output buffer (>= n_img: train and test features stacked)
  const uint8_t* wblob; int blob_bytes, w1_bytes, w2_bytes;   // per candidate: [B1 image | B2 image]
  int shift_mode, nw2;           // layer 2 issued per plane SHIFT (2x2 pooling, 3x3 kernels); number of B2 slots (2 or 3)
  int n_cand, cand_per_cta;
  float* Hout; long long F; float scale;
  int n_layers;
  // layer 1
  int k1, pd1, P1, nph1, Cout1, Cp1, N1, K1, K1p, Pk1, Ho1, Wo1, act1;
  // layer 2
  int k2, pd2, P2, nph2, Cout2, N2, Ho2, Wo2, act2, Wq, Hq, base0, NPOS2;
  int B, NP1, NP1p, T1, NM2, T2, NPB, lg_nslot1, lg_nset1;   // R1 ring slots / E1 warp sets (powers of two)
  // shared-memory offsets (bytes)
  int off_img, off_a1, off_w1, off_w2, off_pl, off_tab1, off_tab2, plane_bytes, plbuf_bytes;
  // TMEM column offsets
  int tm_r1, tm_r2;
};


// barrier slots
enum { W1_FULL = 0, W1_EMPTY = 2, W2_FULL = 4, W2_EMPTY = 7, R1_FULL = 10, R1_EMPTY = 14, PL_FULL = 18, PL_EMPTY = 20,
       R2_FULL = 22, R2_EMPTY = 24, N_BARS = 26 };

// ---- kernel sets -> shared-memory images of the B operands ---------------------------------------------------
// B1: K-major no-swizzle [16-byte K chunk kc][column n][16 B], K index kk = (c*Pk + yy)*Pk + xx over the patch,
//     column n = o*nph1 + (py*P1 + px):  w1[o][c][yy-py][xx-px] where that tap exists, else 0.
// B2: [chunk 0: lo digits | chunk 1: hi digits][tap slot dy*k + (k-1-dx)][column o][16 B = input channel]:
//     w2[o][c][dy][dx] and 64 w2[o][c][dy][dx].  Slots of one kernel row run with dx DEcreasing, so the 2 N2 columns that
//     start at slot (dy, dx) are the taps dx (pool phase px = 0) and dx-1 (px = 1) which read the SAME shifted plane.
struct PrepParams {
  const int8_t* ker; int n_weights; uint8_t* blob; int blob_bytes, w1_bytes, n_layers;
  int k1, P1, nph1, Cout1, N1, K1, K1p, Pk1, Cin1, w1_off;
  int k2, Cout2, N2, w2_off;
  int shift_mode;
};
__global__ void __launch_bounds__(256) xtc_prep_kernel(const PrepParams p) {
  const int cand = blockIdx.y;
  const int8_t* kw = p.ker + (long long)cand * p.n_weights;
  uint8_t* out = p.blob + (long long)cand * p.blob_bytes;
  for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < p.blob_bytes; t += gridDim.x * blockDim.x) {
    int v = 0;
    if (t < p.w1_bytes) {
      const int kb = t & 15, n = (t >> 4) % p.N1, kc = (t >> 4) / p.N1;
      const int kk = kc * 16 + kb;
      const int o = n / p.nph1, ph = n - o * p.nph1;
      if (kk < p.K1 && o < p.Cout1) {
        const int pk2 = p.Pk1 * p.Pk1;
        const int c = kk / pk2, r = kk - c * pk2;
        const int yy = r / p.Pk1, xx = r - yy * p.Pk1;
        const int py = ph / p.P1, px = ph - py * p.P1;
        const int dy = yy - py, dx = xx - px;
        if (dy >= 0 && dy < p.k1 && dx >= 0 && dx < p.k1) v = kw[p.w1_off + ((o * p.Cin1 + c) * p.k1 + dy) * p.k1 + dx];
      }
    } else if (p.n_layers == 2 && p.shift_mode) {
      // per-shift B2 (2x2 pooling, 3x3 kernels): [chunk lo | hi][28 blocks][N2 columns][16 B = input channel].  Blocks 4 s .. 4 s + 3
      // (s = 2 ry + rx, the four plane shifts ry, rx in {0,1} that every pool phase reads): the taps of phases 00, 01, 10, 11,
      // (ry+1, rx+1), (ry+1, rx), (ry, rx+1), (ry, rx).  Blocks 16 + 3 e .. + 2 (e = 2 ry + side; shifts rx = -1 / rx = 2, read by
      // the phases px = 0 / px = 1 only): tap (ry+1, tx), a zero block, tap (ry, tx) with tx = 0 / 2.
      const int u = t - p.w1_bytes;
      const int c = u & 15, o = (u >> 4) % p.N2, blk = ((u >> 4) / p.N2) % 28, half = (u >> 4) / (p.N2 * 28);
      int dy = -1, dx = -1;
      if (blk < 16) {
        const int sft = blk >> 2, q = blk & 3, ry = sft >> 1, rx = sft & 1;
        dy = ry + 1 - (q >> 1); dx = rx + 1 - (q & 1);
      } else {
        const int e = (blk - 16) / 3, q = (blk - 16) % 3, ry = e >> 1, side = e & 1;
        if (q != 1) { dy = ry + (q == 0 ? 1 : 0); dx = side ? 2 : 0; }
      }
      if (dy >= 0 && o < p.Cout2 && c < p.Cout1) {
        v = kw[p.w2_off + (o * p.Cout1 + c) * 9 + dy * 3 + dx];
        if (half) v *= 64;
      }
    } else if (p.n_layers == 2) {
      const int u = t - p.w1_bytes, kk2 = p.k2 * p.k2;
      const int c = u & 15, o = (u >> 4) % p.N2, slot = ((u >> 4) / p.N2) % kk2, half = (u >> 4) / (p.N2 * kk2);
      const int dy = slot / p.k2, dx = p.k2 - 1 - slot % p.k2;      // taps of a row stored with dx DEcreasing
      if (o < p.Cout2 && c < p.Cout1) {
        v = kw[p.w2_off + (o * p.Cout1 + c) * kk2 + dy * p.k2 + dx];
        if (half) v *= 64;
      }
    }
    out[t] = (uint8_t)(int8_t)v;
  }
}

__device__ __forceinline__ int floordiv(int a, int b) { return (a >= 0) ? a / b : -((-a + b - 1) / b); }

// max over NPH adjacent columns for each of the 16 / NPH channels of one 16-column group
template <int NPH>
__device__ __forceinline__ void pool_group(const uint32_t (&r)[16], int* mx) {
#pragma unroll
  for (int q = 0; q < 16 / NPH; ++q) {
    int m = (int)r[q * NPH];
#pragma unroll
    for (int ph = 1; ph < NPH; ++ph) m = max(m, (int)r[q * NPH + ph]);
    mx[q] = m;
  }
}

__device__ __forceinline__ uint32_t bar_addr(const uint64_t* bars, int i) { return tc::smem_u32(bars + i); }

// ---- E1, two layers: R1 -> max-pool -> (relu) -> digits -> phase planes of layer 2 --------------------------------
// tab1[m] = byte offset of pooled position m inside one plane buffer (phase plane + halo-sharing position), -1 = none
// four values -> their low bytes in one word
__device__ __forceinline__ uint32_t pack4(uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  return __byte_perm(__byte_perm(a, b, 0x0040), __byte_perm(c, d, 0x0040), 0x5410);
}

template <int NPH, bool RELU>
__device__ __forceinline__ void e1_two_layer(const XtcParams& p, uint8_t* smem, const uint64_t* bars, uint32_t tmem,
                                             int set, int quad, int lane, int n_cta_cand) {
  constexpr int CPG = 16 / NPH;          // channels per 16-column group
  const uint32_t lane_base = (uint32_t)(quad * 32) << 16;
  // loop invariants in registers (the asm statements' memory clobbers would otherwise re-read the parameters)
  const int lg_slot = p.lg_nslot1, mask = (1 << p.lg_nset1) - 1, smask = (1 << lg_slot) - 1;
  const int T1 = p.T1, N1 = p.N1, npb2 = (p.NPB == 2), nwords = (p.Cp1 + 3) >> 2;
  const int32_t* tab1 = reinterpret_cast<const int32_t*>(smem + p.off_tab1) + quad * 32 + lane;
  const uint32_t taddr0 = tmem + lane_base + p.tm_r1;
  uint8_t* planes0 = smem + p.off_pl;
  const int plbuf_bytes = p.plbuf_bytes, hi_off = p.NPOS2 * 16;
  const uint32_t bar_full0 = bar_addr(bars, R1_FULL), bar_empty0 = bar_addr(bars, R1_EMPTY);
  for (int ci = 0; ci < n_cta_cand; ++ci) {
    const int buf = npb2 ? (ci & 1) : 0;
    const int use = npb2 ? (ci >> 1) : ci;
    bool waited = false;
    for (int t1 = 0; t1 < T1; ++t1) {
      const int n1 = ci * T1 + t1;
      if ((n1 & mask) != set) continue;
      const int slot = n1 & smask;
      const uint32_t taddr = taddr0 + slot * N1;
      tc::mbar_wait(bar_full0 + 8 * slot, (n1 >> lg_slot) & 1);
      tc::tc_fence_after();
      int mx[16];
#pragma unroll
      for (int e = 0; e < 16; ++e) mx[e] = 0;
#pragma unroll
      for (int gb = 0; gb < NPH; gb += 4) {
        if (gb * 16 < N1) {
          uint32_t r[4][16];
#pragma unroll
          for (int q = 0; q < 4; ++q)
            if (gb + q < NPH && (gb + q) * 16 < N1) tc::tmem_ld16(taddr + (gb + q) * 16, r[q]);
          tc::tmem_ld_wait();
#pragma unroll
          for (int q = 0; q < 4; ++q)
            if (gb + q < NPH && (gb + q) * 16 < N1) pool_group<NPH>(r[q], &mx[(gb + q) * CPG]);
        }
      }
      tc::tc_fence_before();
      __syncwarp();
      if (lane == 0) tc::mbar_arrive(bar_empty0 + 8 * slot);               // accumulator slot free again
      if (!waited) { tc::mbar_wait(bar_addr(bars, PL_EMPTY + buf), (use & 1) ^ 1); waited = true; }
      const int32_t off = tab1[t1 * 128];
      if (off >= 0) {
        // v = 64 (v >> 6) + (v & 63): both digits fit an int8; four channels per word, words past the real channels stay 0
        uint32_t lo[4] = {0, 0, 0, 0}, hi[4] = {0, 0, 0, 0};
#pragma unroll
        for (int w = 0; w < 4; ++w) {
          if (w < nwords) {
            int v[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) v[e] = RELU ? max(mx[4 * w + e], 0) : mx[4 * w + e];
            lo[w] = pack4((uint32_t)v[0], (uint32_t)v[1], (uint32_t)v[2], (uint32_t)v[3]) & 0x3f3f3f3fu;
            hi[w] = pack4((uint32_t)(v[0] >> 6), (uint32_t)(v[1] >> 6), (uint32_t)(v[2] >> 6), (uint32_t)(v[3] >> 6));
          }
        }
        uint8_t* dst = planes0 + buf * plbuf_bytes + off;
        *reinterpret_cast<uint4*>(dst) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
        *reinterpret_cast<uint4*>(dst + hi_off) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
      }
    }
    if (!waited) tc::mbar_wait(bar_addr(bars, PL_EMPTY + buf), (use & 1) ^ 1);   // never run ahead of the buffer's phase
    tc::fence_proxy_async();                 // generic-proxy plane writes -> visible to the MMA's async proxy
    __syncwarp();
    if (lane == 0) tc::mbar_arrive(bar_addr(bars, PL_FULL + buf));
  }
}

// ---- E1, single layer: R1 -> max-pool -> (relu) -> scale -> H -------------------------------------------------------
// tab1[m] = b*F + i*Wo + j of pooled position m (flatten C,H,W adds o*Ho*Wo), -1 = none
template <int NPH, bool RELU, bool UNIT>
__device__ __forceinline__ void e1_single(const XtcParams& p, const uint8_t* smem, const uint64_t* bars, uint32_t tmem,
                                          int set, int quad, int lane, int c_begin, int n_cta_cand, long long img0) {
  constexpr int CPG = 16 / NPH;
  const uint32_t lane_base = (uint32_t)(quad * 32) << 16;
  // loop invariants in registers (the asm statements' memory clobbers would otherwise re-read the parameters)
  const int lg_slot = p.lg_nslot1, mask = (1 << p.lg_nset1) - 1, smask = (1 << lg_slot) - 1;
  const int T1 = p.T1, N1 = p.N1, G1 = N1 >> 4, cout1 = p.Cout1;
  const uint32_t hw = (uint32_t)(p.Ho1 * p.Wo1);
  const float scale = p.scale;
  const int32_t* tab1 = reinterpret_cast<const int32_t*>(smem + p.off_tab1) + quad * 32 + lane;
  const uint32_t taddr0 = tmem + lane_base + p.tm_r1;
  const uint32_t bar_full0 = bar_addr(bars, R1_FULL), bar_empty0 = bar_addr(bars, R1_EMPTY);
  const long long cand_stride = p.out_rows * p.F;
  float* Hb = p.Hout + ((long long)c_begin * p.out_rows + img0) * p.F;
  for (int ci = 0; ci < n_cta_cand; ++ci, Hb += cand_stride) {
    for (int t1 = 0; t1 < T1; ++t1) {
      const int n1 = ci * T1 + t1;
      if ((n1 & mask) != set) continue;
      const int slot = n1 & smask;
      const uint32_t taddr = taddr0 + slot * N1;
      tc::mbar_wait(bar_full0 + 8 * slot, (n1 >> lg_slot) & 1);
      tc::tc_fence_after();
      const int32_t off = tab1[t1 * 128];
      uint32_t idx = (uint32_t)(off >= 0 ? off : 0);
      for (int gb = 0; gb < G1; gb += 4) {
        uint32_t r[4][16];
#pragma unroll
        for (int q = 0; q < 4; ++q)
          if (gb + q < G1) tc::tmem_ld16(taddr + (gb + q) * 16, r[q]);
        tc::tmem_ld_wait();
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          if (gb + q < G1) {
            int mx[CPG];
            pool_group<NPH>(r[q], mx);
            if (off >= 0) {
#pragma unroll
              for (int k = 0; k < CPG; ++k) {
                if ((gb + q) * CPG + k < cout1) {
                  const int v = RELU ? max(mx[k], 0) : mx[k];
                  Hb[idx] = UNIT ? (float)v : scale * (float)v;            // flatten C,H,W: channel stride Ho*Wo
                  idx += hw;
                }
              }
            }
          }
        }
      }
      tc::tc_fence_before();
      __syncwarp();
      if (lane == 0) tc::mbar_arrive(bar_empty0 + 8 * slot);
    }
  }
}

// ---- E2: R2 -> max over the pool-phase accumulators -> (relu) -> scale -> H ------------------------------------------
// tab2[m] = b*F + i*Wo2 + j of row m of the halo-sharing output grid, -1 = halo / beyond the batch
template <bool RELU, bool UNIT>
__device__ __forceinline__ void e2_store16(float* __restrict__ Hb, uint32_t idx, uint32_t hw, const int (&mx)[16], int nreal, float scale) {
  if (nreal == 16) {
#pragma unroll
    for (int e = 0; e < 16; ++e) {
      int v = mx[e];
      if (RELU) v = max(v, 0);
      Hb[idx] = UNIT ? (float)v : scale * (float)v;                        // flatten C,H,W: channel stride Ho*Wo
      idx += hw;
    }
  } else {
#pragma unroll
    for (int e = 0; e < 16; ++e) {
      if (e < nreal) {
        int v = mx[e];
        if (RELU) v = max(v, 0);
        Hb[idx] = UNIT ? (float)v : scale * (float)v;
        idx += hw;
      }
    }
  }
}

template <bool RELU, bool UNIT>
__device__ __forceinline__ void e2_run(const XtcParams& p, const uint8_t* smem, const uint64_t* bars, uint32_t tmem, int set,
                                       int quad, int lane, int c_begin, int n_cta_cand, long long img0) {
  const uint32_t lane_base = (uint32_t)(quad * 32) << 16;
  const int32_t* tab2 = reinterpret_cast<const int32_t*>(smem + p.off_tab2);
  const int nph2 = p.nph2, N2 = p.N2, cout2 = p.Cout2, T2 = p.T2;
  const uint32_t hw = (uint32_t)(p.Ho2 * p.Wo2);
  const float scale = p.scale;
  const uint32_t taddr = tmem + lane_base + p.tm_r2 + set * (nph2 * N2);
  const long long cand_stride = p.out_rows * p.F;
  float* Hb = p.Hout + ((long long)c_begin * p.out_rows + img0) * p.F;
  for (int ci = 0; ci < n_cta_cand; ++ci, Hb += cand_stride) {
    for (int t2 = 0; t2 < T2; ++t2) {
      const int n2 = ci * T2 + t2;
      if ((n2 & 1) != set) continue;
      tc::mbar_wait(bar_addr(bars, R2_FULL + set), (n2 >> 1) & 1);
      tc::tc_fence_after();
      const int32_t off = tab2[t2 * 128 + quad * 32 + lane];
      for (int c0 = 0; c0 < cout2; c0 += 16) {
        if (cout2 - c0 <= 4 && nph2 == 4) {
          // tail of up to four channels (configs[1]: 20 = 16 + 4): four-column loads, a quarter of the max / store work
          uint32_t q0[4], q1[4], q2[4], q3[4];
          tc::tmem_ld4(taddr + c0, q0);
          tc::tmem_ld4(taddr + N2 + c0, q1);
          tc::tmem_ld4(taddr + 2 * N2 + c0, q2);
          tc::tmem_ld4(taddr + 3 * N2 + c0, q3);
          tc::tmem_ld_wait();
          if (off >= 0) {
            uint32_t idx = (uint32_t)off + (uint32_t)c0 * hw;
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              if (c0 + e < cout2) {
                int v = max(max((int)q0[e], (int)q1[e]), max((int)q2[e], (int)q3[e]));
                if (RELU) v = max(v, 0);
                Hb[idx] = UNIT ? (float)v : scale * (float)v;
                idx += hw;
              }
            }
          }
          continue;
        }
        int mx[16];
        {
          uint32_t r0[16], r1[16];
          tc::tmem_ld16(taddr + c0, r0);
          if (nph2 > 1) tc::tmem_ld16(taddr + N2 + c0, r1);
          tc::tmem_ld_wait();
#pragma unroll
          for (int e = 0; e < 16; ++e) mx[e] = (nph2 > 1) ? max((int)r0[e], (int)r1[e]) : (int)r0[e];
        }
        for (int ph = 2; ph < nph2; ph += 2) {
          uint32_t r0[16], r1[16];
          tc::tmem_ld16(taddr + ph * N2 + c0, r0);
          tc::tmem_ld16(taddr + (ph + 1) * N2 + c0, r1);
          tc::tmem_ld_wait();
#pragma unroll
          for (int e = 0; e < 16; ++e) mx[e] = max(mx[e], max((int)r0[e], (int)r1[e]));
        }
        if (off >= 0) e2_store16<RELU, UNIT>(Hb, (uint32_t)off + (uint32_t)c0 * hw, hw, mx, min(16, cout2 - c0), scale);
      }
      tc::tc_fence_before();
      __syncwarp();
      if (lane == 0) tc::mbar_arrive(bar_addr(bars, R2_EMPTY + set));
    }
  }
}

// ---- layer-2 MMA issue for one 128-row tile -------------------------------------------------------------------------
// All P2*P2*k*k (phase, tap) MMAs of the tile.  With P2 / K2 known at compile time every plane / shift / tap index
// folds to a constant, so one MMA costs a handful of uniform-datapath instructions (descriptor = base + offset in
// 16-byte units; the sums stay inside the 14-bit address field because every operand lies in shared memory).
template <int P2c, int K2c>
__device__ __forceinline__ void l2_issue_tile(const XtcParams& p, int half, uint32_t d0, uint64_t da0, uint64_t db0, uint32_t idesc2) {
  const int P2 = P2c ? P2c : p.P2, K2 = K2c ? K2c : p.k2;
  const int pd = (K2 - 1) / 2;
  const int plane16 = p.plane_bytes >> 4, n2 = p.N2;
  if constexpr (P2c == 2) {
    // 2x2 pooling: the phases px = 0 (tap dx) and px = 1 (tap dx - 1) of one py read the same shifted plane
    // rx = dx - pd, so one MMA with N = 2 N2 feeds both accumulators (they are adjacent in TMEM and the two taps are
    // adjacent in B2).  Only rx = -pd (px = 0 alone) and rx = pd + 1 (px = 1 alone) stay N = N2.  Per py and dy the
    // pair MMAs go first, so the very first MMA (dy = 0) initialises both accumulators at once.
    const uint32_t idesc_pair = idesc2 + (((uint32_t)n2 >> 3) << 17);     // N field: 2 N2
    const int py = half;                                                  // issuer warp `half` owns pool row py
#pragma unroll
    for (int dy = 0; dy < K2; ++dy) {
      const int ry = py + dy - pd, qy = floordiv(ry, 2), sy = ry - qy * 2;
      const uint32_t d = d0 + (py * 2) * n2;
#pragma unroll
      for (int rx = 1 - pd; rx <= pd; ++rx) {                             // pairs: px = 0 tap rx + pd, px = 1 tap rx + pd - 1
        const int qx = floordiv(rx, 2), sx = rx - qx * 2;
        const uint64_t da = da0 + (uint64_t)(long long)((sy * 2 + sx) * plane16 + qy * p.Wq + qx);
        const uint64_t db = db0 + (uint64_t)((dy * K2 + (K2 - 1 - (rx + pd))) * n2);
        if (tc::elect_one()) tc::mma_i8(d, da, db, idesc_pair, (dy != 0 || rx != 1 - pd) ? 1u : 0u);
      }
      {                                                                   // px = 0 alone: tap dx = 0, rx = -pd
        const int rx = -pd, qx = floordiv(rx, 2), sx = rx - qx * 2;
        const uint64_t da = da0 + (uint64_t)(long long)((sy * 2 + sx) * plane16 + qy * p.Wq + qx);
        const uint64_t db = db0 + (uint64_t)((dy * K2 + (K2 - 1)) * n2);
        if (tc::elect_one()) tc::mma_i8(d, da, db, idesc2, 1u);
      }
      {                                                                   // px = 1 alone: tap dx = K2 - 1, rx = pd + 1
        const int rx = pd + 1, qx = floordiv(rx, 2), sx = rx - qx * 2;
        const uint64_t da = da0 + (uint64_t)(long long)((sy * 2 + sx) * plane16 + qy * p.Wq + qx);
        const uint64_t db = db0 + (uint64_t)((dy * K2) * n2);
        if (tc::elect_one()) tc::mma_i8(d + n2, da, db, idesc2, 1u);
      }
    }
  } else {
  // general pooling: one MMA per (phase, tap); two issuer warps share a tile by pool rows (all of them when P2 == 1)
#pragma unroll
  for (int py = 0; py < P2; ++py)
#pragma unroll
    for (int px = 0; px < P2; ++px) {
      if (P2 > 1 && (py * 2 >= P2) != (half != 0)) continue;
      const uint32_t d = d0 + (py * P2 + px) * n2;
#pragma unroll
      for (int dy = 0; dy < K2; ++dy) {
        const int ry = py + dy - pd, qy = floordiv(ry, P2), sy = ry - qy * P2;
#pragma unroll
        for (int dx = 0; dx < K2; ++dx) {
          const int rx = px + dx - pd, qx = floordiv(rx, P2), sx = rx - qx * P2;
          const int a_off = (sy * P2 + sx) * plane16 + qy * p.Wq + qx;
          const uint64_t da = da0 + (uint64_t)(long long)a_off;
          const uint64_t db = db0 + (uint64_t)((dy * K2 + (K2 - 1 - dx)) * n2);
          if (tc::elect_one()) tc::mma_i8(d, da, db, idesc2, (dy | dx) != 0);
        }
      }
    }
  }
}

// ---- layer-2 MMA issue per plane SHIFT (2x2 pooling, 3x3 kernels) ------------------------------------------------------------
// A conv output of pool phase (py, px) and tap (dy, dx) reads the phase planes shifted by (ry, rx) = (py + dy - 1, px + dx - 1);
// the 36 (phase, tap) pairs share only 16 shifts.  One MMA per shift feeds every phase that reads it -- the accumulators
// of the four phases are adjacent in TMEM (00 | 01 | 10 | 11) and B2 holds the matching taps side by side:
//   4 centre shifts  : all four phases, N = 4 N2                      (64 clk at N2 = 32: tensor-bound)
//   4 top / bottom   : phases 00,01 / 10,11, N = 2 N2, the tap blocks are the second / first half of a centre block
//   4 left / right   : phases 00,10 / 01,11 -- not adjacent: N = 3 N2 with a zero block between them
//   4 corners        : one phase, N = N2, a block of the left / right images
// 16 MMAs and 832 clk per 128 positions instead of 24 and 1056 (operand fetch, profiles/r2_ubench.md); one issuer warp.
__device__ __forceinline__ void l2_issue_shift(const XtcParams& p, uint32_t d0, uint64_t da0, uint64_t db0, uint32_t idesc2) {
  const int plane16 = p.plane_bytes >> 4, n2 = p.N2;
  const uint32_t nf = ((uint32_t)n2 >> 3) << 17;                       // one more N2 in the descriptor's N field
  bool first = true;
#pragma unroll
  for (int pass = 0; pass < 2; ++pass) {             // the centre shifts first: the very first MMA initialises all four accumulators
#pragma unroll
    for (int ry = -1; ry <= 2; ++ry) {
#pragma unroll
      for (int rx = -1; rx <= 2; ++rx) {
        const bool ymid = (ry == 0 || ry == 1), xmid = (rx == 0 || rx == 1);
        if ((ymid && xmid) != (pass == 0)) continue;
        const int qy = floordiv(ry, 2), sy = ry - qy * 2, qx = floordiv(rx, 2), sx = rx - qx * 2;
        const uint64_t da = da0 + (uint64_t)(long long)((sy * 2 + sx) * plane16 + qy * p.Wq + qx);
        const int cy = ry < 0 ? 0 : (ry > 1 ? 1 : ry);                    // row of the nearest centre shift
        int blk, dphase, nmul;
        if (ymid && xmid)      { blk = 4 * (2 * ry + rx); dphase = 0; nmul = 4; }
        else if (xmid)         { blk = 4 * (2 * cy + rx) + (ry < 0 ? 2 : 0); dphase = ry < 0 ? 0 : 2; nmul = 2; }      // top / bottom
        else if (ymid)         { blk = 16 + 3 * (2 * ry + (rx < 0 ? 0 : 1)); dphase = rx < 0 ? 0 : 1; nmul = 3; }      // left / right
        else                   { blk = 16 + 3 * (2 * cy + (rx < 0 ? 0 : 1)) + (ry < 0 ? 2 : 0); dphase = (ry < 0 ? 0 : 2) + (rx < 0 ? 0 : 1); nmul = 1; }
        const uint64_t db = db0 + (uint64_t)(blk * n2);
        const uint32_t idesc = idesc2 + (uint32_t)(nmul - 1) * nf;
        if (tc::elect_one()) tc::mma_i8(d0 + dphase * n2, da, db, idesc, first ? 0u : 1u);
        first = false;
      }
    }
  }
}

// ---- the kernel ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(XT_THREADS, 1) expand_tc_kernel(const XtcParams p) {
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ __align__(8) uint64_t bars[N_BARS];
  __shared__ uint32_t tmem_base_s;
  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = tc::uniform_warp_id();
  const long long img0 = (long long)blockIdx.x * p.B;
  const int nb = (int)min((long long)p.B, p.n_img - img0);         // images really present in this batch
  const int c_begin = blockIdx.y * p.cand_per_cta;
  const int n_cta_cand = min(p.cand_per_cta, p.n_cand - c_begin);
  const uint32_t s_base = tc::smem_u32(smem);
  const int nslot1 = 1 << p.lg_nslot1;
  const int n_e1_warps = 4 << p.lg_nset1;
  const int n_l2_issuers = (p.n_layers == 2 && p.P2 > 1 && !p.shift_mode) ? 2 : 1;     // warps 1 and 18 split a tile's pool phases

  if (tid == 0) {
    for (int i = 0; i < N_BARS; ++i) {
      int cnt = 1;
      if (i >= R1_EMPTY && i < R1_EMPTY + 4) cnt = 4;
      if (i >= R2_EMPTY && i < R2_EMPTY + 2) cnt = 4;
      if (i >= PL_FULL && i < PL_FULL + 2) cnt = n_e1_warps;
      if ((i >= R2_FULL && i < R2_FULL + 2) || (i >= PL_EMPTY && i < PL_EMPTY + 2) || (i >= W2_EMPTY && i < W2_EMPTY + 3)) cnt = n_l2_issuers;
      tc::mbar_init(bar_addr(bars, i), cnt);
    }
    tc::fence_barrier_init();
  }
  if (warp == 0) tc::tmem_alloc(tc::smem_u32(&tmem_base_s), 512);
  // ---- set-up shared by every candidate of this CTA ----
  const int npx = p.H * p.W * p.C;
  {
    const uint8_t* src = p.img + img0 * npx;
    const int total = p.B * npx, have = nb * npx;
    if ((npx & 15) == 0) {          // every image (and so the batch) starts 16-byte aligned
      const uint4* s4 = reinterpret_cast<const uint4*>(src);
      uint4* d4 = reinterpret_cast<uint4*>(smem + p.off_img);
      for (int t = tid; t < total / 16; t += XT_THREADS) d4[t] = (t * 16 < have) ? s4[t] : make_uint4(0, 0, 0, 0);
    } else {
      for (int t = tid; t < total; t += XT_THREADS) smem[p.off_img + t] = (t < have) ? src[t] : (uint8_t)0;
    }
    if (p.n_layers == 2) {
      uint4* pl = reinterpret_cast<uint4*>(smem + p.off_pl);
      const int n16 = p.NPB * p.plbuf_bytes / 16;
      for (int t = tid; t < n16; t += XT_THREADS) pl[t] = make_uint4(0, 0, 0, 0);
      // tab2: row m of the halo-sharing output grid -> b*F + i2*Wo2 + j2
      int32_t* tab2 = reinterpret_cast<int32_t*>(smem + p.off_tab2);
      for (int m = tid; m < p.T2 * 128; m += XT_THREADS) {
        const int b = m / (p.Hq * p.Wq), rem = m - b * (p.Hq * p.Wq);
        const int i2 = rem / p.Wq, j2 = rem - i2 * p.Wq;
        const bool ok = (m < p.NM2) && (b < nb) && (i2 < p.Ho2) && (j2 < p.Wo2);
        tab2[m] = ok ? (int32_t)(b * p.F + i2 * p.Wo2 + j2) : -1;
      }
    }
    // tab1: pooled layer-1 position m -> plane offset (two layers) or b*F + i1*Wo1 + j1 (single layer)
    int32_t* tab1 = reinterpret_cast<int32_t*>(smem + p.off_tab1);
    const int plane1 = p.Ho1 * p.Wo1;
    for (int m = tid; m < p.NP1p; m += XT_THREADS) {
      int32_t v = -1;
      if (m < p.NP1) {
        const int b = m / plane1, rem = m - b * plane1;
        const int i1 = rem / p.Wo1, j1 = rem - i1 * p.Wo1;
        if (p.n_layers == 2) {
          const int sy = i1 % p.P2, sx = j1 % p.P2;
          const int pos = p.base0 + (b * p.Hq + i1 / p.P2) * p.Wq + j1 / p.P2;
          v = (sy * p.P2 + sx) * p.plane_bytes + pos * 16;
        } else if (b < nb) {
          v = (int32_t)(b * p.F + i1 * p.Wo1 + j1);
        }
      }
      tab1[m] = v;
    }
  }
  __syncthreads();          // images in shared memory
  {
    // A1: [16-byte K chunk][pooled position][16 B]; K index = (c*Pk + yy)*Pk + xx over the (P+k-1)^2 x Cin patch
    const int plane1 = p.Ho1 * p.Wo1, pk2 = p.Pk1 * p.Pk1;
    const int nchunk = p.K1p / 16;
    for (int t = tid; t < p.NP1p * nchunk; t += XT_THREADS) {
      const int m = t % p.NP1p, kc = t / p.NP1p;
      uint32_t w[4] = {0, 0, 0, 0};
      if (m < p.NP1) {
        const int b = m / plane1, rem = m - b * plane1;
        const int i1 = rem / p.Wo1, j1 = rem - i1 * p.Wo1;
        const uint8_t* im = smem + p.off_img + b * npx;
        const int y0 = p.P1 * i1 - p.pd1, x0 = p.P1 * j1 - p.pd1;
#pragma unroll 4
        for (int e = 0; e < 16; ++e) {
          const int kk = kc * 16 + e;
          if (kk < p.K1) {
            const int c = kk / pk2, r = kk - c * pk2;
            const int yy = r / p.Pk1, xx = r - yy * p.Pk1;
            const int y = y0 + yy, x = x0 + xx;
            if (y >= 0 && y < p.H && x >= 0 && x < p.W) w[e >> 2] |= (uint32_t)im[(y * p.W + x) * p.C + c] << (8 * (e & 3));
          }
        }
      }
      *reinterpret_cast<uint4*>(smem + p.off_a1 + (kc * p.NP1p + m) * 16) = make_uint4(w[0], w[1], w[2], w[3]);
    }
  }
  tc::fence_proxy_async();      // generic-proxy writes (A1, zeroed planes) -> visible to the MMA's async proxy
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t tmem = tmem_base_s;

  if (warp == 0) {
    // ===== layer-1 issuer =====
    const uint32_t idesc1 = tc::idesc_i8(128, p.N1, 0, 1, 0, 0);     // u8 pixels x s8 weights, K-major both
    const int nks = p.K1p / 32;
    const uint32_t lbo_a = (uint32_t)p.NP1p * 16, lbo_b = (uint32_t)p.N1 * 16;
    // loop invariants: descriptors are "base + offset in 16-byte units" (this warp's latency per tile is what keeps
    // the E1 warps fed, so nothing is rebuilt inside the tile loop)
    const uint64_t da_base = tc::smem_desc(s_base + p.off_a1, lbo_a, 128, tc::LAYOUT_NONE);
    const uint64_t db_base = tc::smem_desc(s_base + p.off_w1, lbo_b, 128, tc::LAYOUT_NONE);
    const uint32_t a_ks = 2 * p.NP1p, b_ks = 2 * p.N1, b_slot = p.w1_bytes >> 4, d_base = tmem + p.tm_r1, n1cols = p.N1;
    const int T1 = p.T1, lg = p.lg_nslot1;
    const uint32_t bar_full0 = bar_addr(bars, R1_FULL), bar_empty0 = bar_addr(bars, R1_EMPTY);
    int n1 = 0;
    for (int ci = 0; ci < n_cta_cand; ++ci) {
      if (ci == 0 && tc::elect_one()) {
        tc::mbar_arrive_expect_tx(bar_addr(bars, W1_FULL), p.w1_bytes);
        tc::bulk_load(s_base + p.off_w1, p.wblob + (long long)c_begin * p.blob_bytes, p.w1_bytes, bar_addr(bars, W1_FULL));
      }
      if (ci + 1 < n_cta_cand) {          // stage the next candidate's B1 while this one computes
        const int slot = (ci + 1) & 1, use = (ci + 1) >> 1;
        tc::mbar_wait(bar_addr(bars, W1_EMPTY + slot), (use & 1) ^ 1);
        if (tc::elect_one()) {
          tc::mbar_arrive_expect_tx(bar_addr(bars, W1_FULL + slot), p.w1_bytes);
          tc::bulk_load(s_base + p.off_w1 + slot * p.w1_bytes, p.wblob + (long long)(c_begin + ci + 1) * p.blob_bytes, p.w1_bytes,
                        bar_addr(bars, W1_FULL + slot));
        }
      }
      tc::mbar_wait(bar_addr(bars, W1_FULL + (ci & 1)), (ci >> 1) & 1);
      const uint64_t db_c = db_base + (uint64_t)((ci & 1) * b_slot);
      for (int t1 = 0; t1 < T1; ++t1, ++n1) {
        const int slot = n1 & (nslot1 - 1);
        tc::mbar_wait(bar_empty0 + 8 * slot, ((n1 >> lg) & 1) ^ 1);
        tc::tc_fence_after();
        const uint32_t d = d_base + slot * n1cols;
        const uint64_t da_t = da_base + (uint64_t)(t1 * 128);
        for (int ks = 0; ks < nks; ++ks)
          if (tc::elect_one()) tc::mma_i8(d, da_t + (uint64_t)(ks * a_ks), db_c + (uint64_t)(ks * b_ks), idesc1, ks > 0);
        if (tc::elect_one()) tc::mma_commit(bar_full0 + 8 * slot);
      }
      if (tc::elect_one()) tc::mma_commit(bar_addr(bars, W1_EMPTY + (ci & 1)));
      __syncwarp();
    }
  } else if (warp == 1 || warp == XT_WARPS - 1) {
    // ===== layer-2 issuers =====
    const int half = (warp == 1) ? 0 : 1;
    if (p.n_layers == 2 && half < n_l2_issuers) {
      const uint32_t idesc2 = tc::idesc_i8(128, p.N2, 1, 1, 0, 0);
      const uint32_t lbo_a = (uint32_t)p.NPOS2 * 16, lbo_b = (uint32_t)((p.shift_mode ? 28 : p.k2 * p.k2) * p.N2) * 16;   // digit-chunk strides
      const int nw2 = p.nw2;
      const int acc_cols = p.nph2 * p.N2;
      int n2 = 0;
      for (int ci = 0; ci < n_cta_cand; ++ci) {
        if (half == 0 && ci == 0 && tc::elect_one()) {
          tc::mbar_arrive_expect_tx(bar_addr(bars, W2_FULL), p.w2_bytes);
          tc::bulk_load(s_base + p.off_w2, p.wblob + (long long)c_begin * p.blob_bytes + p.w1_bytes, p.w2_bytes, bar_addr(bars, W2_FULL));
        }
        if (half == 0 && ci + 1 < n_cta_cand) {
          const int slot = (ci + 1) % nw2, use = (ci + 1) / nw2;
          tc::mbar_wait(bar_addr(bars, W2_EMPTY + slot), (use & 1) ^ 1);
          if (tc::elect_one()) {
            tc::mbar_arrive_expect_tx(bar_addr(bars, W2_FULL + slot), p.w2_bytes);
            tc::bulk_load(s_base + p.off_w2 + slot * p.w2_bytes, p.wblob + (long long)(c_begin + ci + 1) * p.blob_bytes + p.w1_bytes,
                          p.w2_bytes, bar_addr(bars, W2_FULL + slot));
          }
        }
        const int wslot = ci % nw2;
        tc::mbar_wait(bar_addr(bars, W2_FULL + wslot), (ci / nw2) & 1);
        const int buf = (p.NPB == 2) ? (ci & 1) : 0;
        const int use = (p.NPB == 2) ? (ci >> 1) : ci;
        tc::mbar_wait(bar_addr(bars, PL_FULL + buf), use & 1);
        const uint32_t pl_base = s_base + p.off_pl + buf * p.plbuf_bytes;
        const uint32_t b_base = s_base + p.off_w2 + wslot * p.w2_bytes;
        for (int t2 = 0; t2 < p.T2; ++t2, ++n2) {
          const int slot = n2 & 1;
          tc::mbar_wait(bar_addr(bars, R2_EMPTY + slot), ((n2 >> 1) & 1) ^ 1);
          tc::tc_fence_after();
          const uint32_t d0 = tmem + p.tm_r2 + slot * acc_cols;
          const uint32_t row0 = (uint32_t)(p.base0 + t2 * 128) * 16;
          const uint64_t da0 = tc::smem_desc(pl_base + row0, lbo_a, 128, tc::LAYOUT_NONE);
          const uint64_t db0 = tc::smem_desc(b_base, lbo_b, 128, tc::LAYOUT_NONE);
          if (p.shift_mode) l2_issue_shift(p, d0, da0, db0, idesc2);
          else if (p.P2 == 2 && p.k2 == 3) l2_issue_tile<2, 3>(p, half, d0, da0, db0, idesc2);
          else if (p.P2 == 1 && p.k2 == 3) l2_issue_tile<1, 3>(p, half, d0, da0, db0, idesc2);
          else l2_issue_tile<0, 0>(p, half, d0, da0, db0, idesc2);
          if (tc::elect_one()) tc::mma_commit(bar_addr(bars, R2_FULL + slot));
          __syncwarp();
        }
        if (tc::elect_one()) {
          tc::mma_commit(bar_addr(bars, PL_EMPTY + buf));
          tc::mma_commit(bar_addr(bars, W2_EMPTY + wslot));
        }
        __syncwarp();
      }
    }
  } else if (warp < 2 + n_e1_warps) {
    const int set = (warp - 2) >> 2, quad = warp & 3;
    if (p.n_layers == 2) {
      const bool relu1 = p.act1 == LBCNN_ACT_RELU;
      if (p.nph1 == 4 && !relu1) e1_two_layer<4, false>(p, smem, bars, tmem, set, quad, lane, n_cta_cand);
      else if (p.nph1 == 4) e1_two_layer<4, true>(p, smem, bars, tmem, set, quad, lane, n_cta_cand);
      else if (p.nph1 == 1 && !relu1) e1_two_layer<1, false>(p, smem, bars, tmem, set, quad, lane, n_cta_cand);
      else if (p.nph1 == 1) e1_two_layer<1, true>(p, smem, bars, tmem, set, quad, lane, n_cta_cand);
      else if (!relu1) e1_two_layer<16, false>(p, smem, bars, tmem, set, quad, lane, n_cta_cand);
      else e1_two_layer<16, true>(p, smem, bars, tmem, set, quad, lane, n_cta_cand);
    } else {
      // the search driver's case (no relu, scale 1) is specialised; everything else takes the general instantiation
      const bool plain = p.act1 != LBCNN_ACT_RELU && p.scale == 1.0f;
#define XT_E1S(NPH)                                                                                                      \
  do {                                                                                                                   \
    if (plain) e1_single<NPH, false, true>(p, smem, bars, tmem, set, quad, lane, c_begin, n_cta_cand, img0); \
    else if (p.act1 == LBCNN_ACT_RELU)                                                                                   \
      e1_single<NPH, true, false>(p, smem, bars, tmem, set, quad, lane, c_begin, n_cta_cand, img0);         \
    else e1_single<NPH, false, false>(p, smem, bars, tmem, set, quad, lane, c_begin, n_cta_cand, img0);     \
  } while (0)
      if (p.nph1 == 1) XT_E1S(1);
      else if (p.nph1 == 4) XT_E1S(4);
      else XT_E1S(16);
#undef XT_E1S
    }
  } else if (p.n_layers == 2) {
    const int set = (warp - 2 - n_e1_warps) >> 2, quad = warp & 3;
    const bool relu = p.act2 == LBCNN_ACT_RELU, unit = p.scale == 1.0f;
    if (relu) {
      if (unit) e2_run<true, true>(p, smem, bars, tmem, set, quad, lane, c_begin, n_cta_cand, img0);
      else e2_run<true, false>(p, smem, bars, tmem, set, quad, lane, c_begin, n_cta_cand, img0);
    } else {
      if (unit) e2_run<false, true>(p, smem, bars, tmem, set, quad, lane, c_begin, n_cta_cand, img0);
      else e2_run<false, false>(p, smem, bars, tmem, set, quad, lane, c_begin, n_cta_cand, img0);
    }
  }
  tc::tc_fence_before();
  __syncthreads();
  if (warp == 0) { tc::tc_fence_after(); tc::tmem_dealloc(tmem, 512); }
}

}  // namespace

// ---- host side ------------------------------------------------------------------------------------------------------------
// Is the architecture inside the tensor-core kernel's envelope?  Fills the launch parameters if so.
static bool plan_xtc(const lbcnn_handle_s* h, const ArchShape& s, bool has_bias, XtcParams* q, size_t* smem_bytes) {
  if (has_bias || s.n_layers < 1 || s.n_layers > 2) return false;
  for (int l = 0; l < s.n_layers; ++l) {
    const LayerShape& L = s.L[l];
    if (L.conv_type != LBCNN_CONV_FULL || L.pp != 0 || L.cover != 0 || L.pk != L.ps) return false;
    if (L.pk != 1 && L.pk != 2 && L.pk != 4) return false;
    if (L.hin % L.pk != 0 || L.win % L.pk != 0) return false;
  }
  XtcParams p{};
  const LayerShape& A = s.L[0];
  p.H = A.hin; p.W = A.win; p.C = A.cin; p.n_layers = s.n_layers;
  p.k1 = A.k; p.pd1 = (A.k - 1) / 2; p.P1 = A.pk; p.nph1 = A.pk * A.pk; p.Cout1 = A.cout;
  p.Pk1 = A.pk + A.k - 1; p.K1 = p.Pk1 * p.Pk1 * A.cin; p.K1p = (p.K1 + 31) / 32 * 32;
  p.Ho1 = A.hout; p.Wo1 = A.wout; p.act1 = A.act;
  const int cpg = p.nph1 >= 16 ? 1 : 16 / p.nph1;                 // channels per 16-column group
  p.Cp1 = (p.Cout1 + cpg - 1) / cpg * cpg;
  p.N1 = p.Cp1 * p.nph1;
  if (p.N1 > 256 || p.K1p > 256) return false;
  p.w1_bytes = p.K1p * p.N1;
  int halo = 0;
  if (s.n_layers == 2) {
    const LayerShape& Bq = s.L[1];
    if (p.Cout1 > 16 || 255LL * A.k * A.k * A.cin > 8191) return false;   // 16 channels per K chunk; two int8 digits
    p.k2 = Bq.k; p.pd2 = (Bq.k - 1) / 2; p.P2 = Bq.pk; p.nph2 = Bq.pk * Bq.pk; p.Cout2 = Bq.cout;
    p.Ho2 = Bq.hout; p.Wo2 = Bq.wout; p.act2 = Bq.act;
    p.N2 = (p.Cout2 + 15) / 16 * 16;
    if (p.N2 > 256) return false;
    // two E1 warp sets; each owns two R1 accumulator slots when TMEM has room (so the next tile's MMA is done early)
    p.lg_nset1 = 1; p.lg_nslot1 = (4 * p.N1 + 2 * p.nph2 * p.N2 <= 512) ? 2 : 1;
    p.tm_r1 = 0; p.tm_r2 = (1 << p.lg_nslot1) * p.N1;
    if (p.tm_r2 + 2 * p.nph2 * p.N2 > 512) return false;
    // 2x2 pooling with 3x3 kernels: one MMA per plane shift (l2_issue_shift) -- B2 then holds 28 tap blocks instead of 9
    p.shift_mode = (p.P2 == 2 && p.k2 == 3 && 4 * p.N2 <= 256) ? 1 : 0;
    p.w2_bytes = (p.shift_mode ? 28 : p.k2 * p.k2) * p.N2 * 32;
    const int hq = (p.pd2 + p.P2 - 1) / p.P2, qmax = (p.P2 - 1 + p.pd2) / p.P2;
    halo = hq > qmax ? hq : qmax;
    // Row pitch and first row of the halo-sharing grid.  A shifted operand whose start is not a multiple of 8 rows
    // (128 B) makes every 8-row core matrix straddle two shared-memory lines and the MMA read it in twice the
    // wavefronts, so align the pitch when that costs few extra rows and always align the first row: the taps with
    // no horizontal shift (two thirds of them) then read aligned operands.
    p.Wq = p.Wo2 + halo;
    if (p.Wq % 8 != 0 && (p.Wq + 7) / 8 * 8 * 7 <= p.Wq * 8) p.Wq = (p.Wq + 7) / 8 * 8;
    p.Hq = p.Ho2 + halo; p.base0 = (halo * p.Wq + halo + 7) / 8 * 8;
  } else {
    p.tm_r1 = 0; p.lg_nslot1 = (4 * p.N1 <= 512) ? 2 : 1; p.lg_nset1 = p.lg_nslot1;
    p.w2_bytes = 0;
  }
  p.blob_bytes = p.w1_bytes + p.w2_bytes;
  // images per CTA: the batch size (<= 8) whose 128-row tiles are best filled, within the shared-memory limit
  const int npx = p.H * p.W * p.C;
  const size_t limit = (size_t)h->max_smem_optin;
  double best_score = -1.0; XtcParams best{}; size_t best_smem = 0;
  for (int B = 1; B <= 8; ++B) {
    XtcParams t = p;
    t.B = B; t.NP1 = B * p.Ho1 * p.Wo1; t.T1 = (t.NP1 + 127) / 128; t.NP1p = t.T1 * 128;
    if ((long long)t.NP1p * 16 >= (1 << 18)) break;               // descriptor leading-offset field
    int off = 0;
    auto take = [&](int bytes) { int o = off; off += (bytes + 127) / 128 * 128; return o; };
    t.off_img = take(B * npx);
    t.off_a1 = take(t.NP1p * t.K1p);
    t.off_w1 = take(2 * p.w1_bytes);
    t.off_tab1 = take(t.NP1p * 4);
    double score = (double)t.NP1 / t.NP1p;
    for (int npb = 2; npb >= 1; --npb) {
      XtcParams u = t; int off2 = off;
      auto take2 = [&](int bytes) { int o = off2; off2 += (bytes + 127) / 128 * 128; return o; };
      if (s.n_layers == 2) {
        u.NM2 = B * p.Hq * p.Wq; u.T2 = (u.NM2 + 127) / 128;
        u.NPOS2 = (p.base0 + u.T2 * 128 + halo * p.Wq + halo + 8 + 7) / 8 * 8;
        if (u.NPOS2 * 16 >= (1 << 18)) break;
        u.plane_bytes = 2 * u.NPOS2 * 16;
        u.plbuf_bytes = p.nph2 * u.plane_bytes;
        u.NPB = npb;
        u.nw2 = p.shift_mode ? 2 : 3;                                // the per-shift image is 3x larger: two slots
        u.off_w2 = take2(u.nw2 * p.w2_bytes);
        u.off_tab2 = take2(u.T2 * 128 * 4);
        u.off_pl = take2(npb * u.plbuf_bytes);
        score = 0.3 * t.NP1 / t.NP1p + 0.7 * u.NM2 / (u.T2 * 128.0);
        if (npb == 1) score *= 0.8;                                // single plane buffer: less overlap
      } else {
        u.NPB = 1;
        if (npb == 1) break;
      }
      if ((size_t)off2 + 1024 > limit) continue;
      score += 0.002 * B;                                          // ties: larger batches amortise the set-up
      if (score > best_score) { best_score = score; best = u; best_smem = (size_t)off2; }
      break;
    }
  }
  if (best_score < 0.0) return false;
  *q = best; *smem_bytes = best_smem;
  return true;
}

bool lb_expand_tc_usable(const lbcnn_handle_s* h, const ArchShape& s, bool has_bias) {
  XtcParams q; size_t sm;
  return plan_xtc(h, s, has_bias, &q, &sm);
}

// bytes of caller workspace the tensor-core expander needs for n_cand candidates: the +-1 kernel sets re-laid-out as the
// shared-memory images of the B operands (0 when the architecture takes the SIMT kernel)
size_t lb_expand_tc_ws_bytes(const lbcnn_handle_s* h, const ArchShape& s, bool has_bias, int n_cand) {
  XtcParams q; size_t sm;
  if (!plan_xtc(h, s, has_bias, &q, &sm)) return 0;
  return (size_t)lb_align_up((int64_t)n_cand * q.blob_bytes, 256);
}

int lb_launch_expand_tc(lbcnn_handle_s* h, const ArchShape& s, float feature_scale, const uint8_t* d_images, int64_t n,
                        const int8_t* d_kernels, int n_cand, float* d_H, void* xw, size_t xw_bytes, cudaStream_t st,
                        bool prepared, int64_t out_rows) {
  XtcParams p; size_t smem = 0;
  if (!plan_xtc(h, s, false, &p, &smem)) return LBCNN_ERR_INVALID_ARCH;
  if (n_cand > 65535) return LBCNN_ERR_INVALID_ARG;
  // scratch for the re-laid-out kernel sets comes from the caller's workspace (never a hidden allocation)
  const size_t need = (size_t)n_cand * p.blob_bytes;
  if (!xw || xw_bytes < need) return LBCNN_ERR_WORKSPACE;
  LbPhase ph(h, LBCNN_PHASE_EXPAND, st);
  if (!prepared) {
    PrepParams w{};
    w.ker = d_kernels; w.n_weights = (int)s.n_weights; w.blob = reinterpret_cast<uint8_t*>(xw);
    w.blob_bytes = p.blob_bytes; w.w1_bytes = p.w1_bytes; w.n_layers = p.n_layers;
    w.k1 = p.k1; w.P1 = p.P1; w.nph1 = p.nph1; w.Cout1 = p.Cout1; w.N1 = p.N1; w.K1 = p.K1; w.K1p = p.K1p; w.Pk1 = p.Pk1;
    w.Cin1 = p.C; w.w1_off = (int)s.L[0].w_off;
    if (p.n_layers == 2) { w.k2 = p.k2; w.Cout2 = p.Cout2; w.N2 = p.N2; w.w2_off = (int)s.L[1].w_off; w.shift_mode = p.shift_mode; }
    dim3 grid((unsigned)((p.blob_bytes + 1023) / 1024 < 1 ? 1 : (p.blob_bytes + 1023) / 1024), (unsigned)n_cand);
    xtc_prep_kernel<<<grid, 256, 0, st>>>(w);
    h->launches += 1;
    LB_CUDA_OK(cudaGetLastError());
  }
  p.img = d_images; p.n_img = n; p.wblob = reinterpret_cast<const uint8_t*>(xw); p.n_cand = n_cand;
  p.Hout = d_H; p.F = s.F; p.scale = feature_scale; p.out_rows = out_rows > 0 ? out_rows : n;
  const long long batches = (n + p.B - 1) / p.B;
  // candidates per CTA: as many as possible (they share the staged images and A1) while the grid still
  // covers the SMs about four times over
  int cpc = n_cand;
  const long long want = 4LL * h->n_sm;
  while (cpc > 8 && batches * ((n_cand + cpc - 1) / cpc) < want) cpc = (cpc + 1) / 2;
  p.cand_per_cta = cpc;
  const int gy = (n_cand + cpc - 1) / cpc;
  if (batches > 2147483647LL || gy > 65535) return LBCNN_ERR_INVALID_ARG;
  // one CTA per SM (it owns all 512 TMEM columns): ask for more than half of the SM's shared memory
  if (smem < 120 * 1024) smem = 120 * 1024;
  LB_CUDA_OK(cudaFuncSetAttribute(expand_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  dim3 grid((unsigned)batches, (unsigned)gy);
  expand_tc_kernel<<<grid, XT_THREADS, smem, st>>>(p);
  h->launches += 1;
  LB_CUDA_OK(cudaGetLastError());
  return LBCNN_OK;
}
