// expand_tc.cu -- K1 on the tensor pipe: the LB-CNN expander for FULL convolutions with
// non-overlapping pooling, as exact integer implicit GEMMs on tcgen05.mma kind::i8 (int32 accumulators in TMEM).
//
// Layer 1 (Cin = 1..3 channels of uint8 pixels): explicit im2col rows [position][k*k*Cin -> 32 bytes] built in
// shared memory, one set of rows per POOL PHASE (py,px); u8 x s8 -> s32 MMAs with M = 128 pooled positions,
// N = 16 output channels, K = 32.  The pool is then an element-wise max over the P*P phase accumulators in the
// SAME TMEM lane -- no shuffles ("Nonlinearity achieved in Max-pool").
// Layer 2 (Cin = layer-1 channels, values up to +-8159): the pooled layer-1 map is written to shared memory
// as balanced radix-64 digits v = lo + 64 hi (both int8), split into P*P phase planes
// plane[sy][sx](i,j) = a[P i + sy][P j + sx] with a shared zero halo.  For output phase (py,px) and tap (dy,dx)
// the A operand is a plane shifted by a constant number of positions, i.e. just a different start address of a
// K-major no-swizzle descriptor ("tap-shifted implicit GEMM"): 9 taps accumulate into one TMEM accumulator,
// weights are +-1 (lo digits) and +-64 (hi digits) in the same int8 B operand, so the int32 result is the exact
// convolution.  Pool = max over the phase accumulators again; flatten C,H,W; one multiply by feature_scale.
//
// CTA = a batch of B images x a range of candidates, 128 threads (thread t owns TMEM lane t), thread 0 issues
// the MMAs; tcgen05.commit -> mbarrier hands accumulators to the epilogue.  Two CTAs are resident per SM
// (<= 256 TMEM columns, ~100 KB shared memory each) so one CTA's epilogue overlaps the other's MMAs.
// Anything outside this kernel's envelope (depthwise, overlapping / padded / cover_all pooling, bias, three
// layers, wide layers) takes the exact SIMT kernel in expand.cu.
#include "internal.h"
#include "tc_common.cuh"

namespace {

struct XtcParams {
  const uint8_t* img; long long n_img; int H, W, C;
  const int8_t* ker; int n_weights; int n_cand, cand_per_cta;
  float* Hout; long long F; float scale;
  int n_layers;
  // layer 1
  int k1, pd1, P1, Cout1, K1, K1p, Ho1, Wo1, act1, w1_off;
  // layer 2
  int k2, pd2, P2, Cout2, Ho2, Wo2, act2, w2_off, Wq, Hq, base0, NPOS2, N2;
  int B, NP1, T1, NM2, T2, cache;
  // shared-memory offsets (bytes)
  int off_img, off_w1, off_w2, off_col, off_pl, col_slot_bytes, plane_bytes;
};

__device__ __forceinline__ int floordiv(int a, int b) { return (a >= 0) ? a / b : -((-a + b - 1) / b); }

__global__ void __launch_bounds__(128, 2) expand_tc_kernel(const XtcParams p) {
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ __align__(8) uint64_t bar;
  __shared__ uint32_t tmem_base_s;
  const int tid = threadIdx.x, warp = tid >> 5;
  const long long img0 = (long long)blockIdx.x * p.B;
  const int nb = (int)min((long long)p.B, p.n_img - img0);         // images really present in this batch
  const int c_begin = blockIdx.y * p.cand_per_cta;
  const int c_end = min(c_begin + p.cand_per_cta, p.n_cand);
  const uint32_t s_base = tc::smem_u32(smem);
  const uint32_t bar_a = tc::smem_u32(&bar);

  if (tid == 0) { tc::mbar_init(bar_a, 1); tc::fence_barrier_init(); }
  __syncwarp();
  if (warp == 0) tc::tmem_alloc(tc::smem_u32(&tmem_base_s), 256);
  // raw images of the batch -> shared memory (zero for images beyond n_img); zero the layer-2 planes once
  {
    const int npx = p.H * p.W * p.C;
    const uint8_t* src = p.img + img0 * npx;
    for (int t = tid; t < p.B * npx; t += 128) smem[p.off_img + t] = (t < nb * npx) ? src[t] : (uint8_t)0;
    if (p.n_layers == 2) {
      uint4* pl = reinterpret_cast<uint4*>(smem + p.off_pl);
      const int n16 = p.P2 * p.P2 * p.plane_bytes / 16;
      for (int t = tid; t < n16; t += 128) pl[t] = make_uint4(0, 0, 0, 0);
    }
  }
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t tmem = tmem_base_s;
  const uint32_t lane_base = (uint32_t)(warp * 32) << 16;
  uint32_t parity = 0;

  constexpr uint32_t IDESC1 = tc::idesc_i8(128, 16, 0, 1, 0, 0);   // u8 pixels x s8 weights, K-major both
  const uint32_t idesc2 = tc::idesc_i8(128, p.N2, 1, 1, 0, 0);
  const int nph1 = p.P1 * p.P1;
  const int plane1 = p.Ho1 * p.Wo1;

  for (int cand = c_begin; cand < c_end; ++cand) {
    const int8_t* kw = p.ker + (long long)cand * p.n_weights;
    // ---- weights of this candidate -> B operands (K-major, no swizzle: [16-byte K chunk][row][16 B]) ----
    {
      // layer 1: row o (16 rows), K index = (c*k + dy)*k + dx -- the kernel set's own order
      for (int t = tid; t < 16 * p.K1p; t += 128) {
        const int o = t / p.K1p, kk = t % p.K1p;
        const int8_t v = (o < p.Cout1 && kk < p.K1) ? kw[p.w1_off + o * p.K1 + kk] : (int8_t)0;
        smem[p.off_w1 + (kk >> 4) * 256 + o * 16 + (kk & 15)] = (uint8_t)v;
      }
      if (p.n_layers == 2) {
        // layer 2, per tap: rows o (N2), chunk 0 = +-1 on the lo digits of channel c, chunk 1 = +-64 on the hi digits
        const int kk2 = p.k2 * p.k2, cin2 = p.Cout1;
        for (int t = tid; t < kk2 * p.N2 * 16; t += 128) {
          const int c = t & 15, o = (t >> 4) % p.N2, tap = (t >> 4) / p.N2;
          int v = 0;
          if (o < p.Cout2 && c < cin2) v = kw[p.w2_off + (o * cin2 + c) * kk2 + tap];
          uint8_t* dst = smem + p.off_w2 + tap * (p.N2 * 32) + o * 16 + c;
          dst[0] = (uint8_t)(int8_t)v;
          dst[p.N2 * 16] = (uint8_t)(int8_t)(64 * v);
        }
      }
    }
    // ---- layer 1: tiles of 128 pooled positions ----
    for (int t1 = 0; t1 < p.T1; ++t1) {
      const int slot = p.cache ? t1 : 0;
      const int m1 = t1 * 128 + tid;
      const bool in_range = m1 < p.NP1;
      const int b = in_range ? m1 / plane1 : 0;
      const int rem = in_range ? m1 - b * plane1 : 0;
      const int i1 = rem / p.Wo1, j1 = rem - i1 * p.Wo1;
      if (!p.cache || cand == c_begin) {
        // im2col row of this thread's position for every pool phase: K1p bytes = k*k*Cin pixels, zero padded
        const uint8_t* im = smem + p.off_img + b * (p.H * p.W * p.C);
        for (int ph = 0; ph < nph1; ++ph) {
          const int py = ph / p.P1, px = ph - py * p.P1;
          const int y0 = p.P1 * i1 + py - p.pd1, x0 = p.P1 * j1 + px - p.pd1;
          uint8_t* dst = smem + p.off_col + slot * p.col_slot_bytes + ph * (p.K1p * 128) + tid * 16;
          for (int q = 0; q < p.K1p / 16; ++q) {
            uint32_t w[4] = {0, 0, 0, 0};
            if (in_range) {
#pragma unroll 4
              for (int e = 0; e < 16; ++e) {
                const int kk = q * 16 + e;
                if (kk < p.K1) {
                  const int c = kk / (p.k1 * p.k1), r2 = kk - c * (p.k1 * p.k1);
                  const int dy = r2 / p.k1, dx = r2 - dy * p.k1;
                  const int y = y0 + dy, x = x0 + dx;
                  if (y >= 0 && y < p.H && x >= 0 && x < p.W)
                    w[e >> 2] |= (uint32_t)im[(y * p.W + x) * p.C + c] << (8 * (e & 3));
                }
              }
            }
            *reinterpret_cast<uint4*>(dst + q * 2048) = make_uint4(w[0], w[1], w[2], w[3]);
          }
        }
      }
      tc::fence_proxy_async();      // generic-proxy smem writes (im2col, weights, planes) -> visible to the MMA
      tc::tc_fence_before();
      __syncthreads();
      if (tid == 0) {
        tc::tc_fence_after();
        for (int ph = 0; ph < nph1; ++ph) {
          const uint32_t a0 = s_base + p.off_col + slot * p.col_slot_bytes + ph * (p.K1p * 128);
          for (int ks = 0; ks < p.K1p / 32; ++ks) {
            const uint64_t da = tc::smem_desc(a0 + ks * 4096, 2048, 128, tc::LAYOUT_NONE);
            const uint64_t db = tc::smem_desc(s_base + p.off_w1 + ks * 512, 256, 128, tc::LAYOUT_NONE);
            tc::mma_i8(tmem + ph * 16, da, db, IDESC1, ks > 0);
          }
        }
        tc::mma_commit(bar_a);
      }
      tc::mbar_wait(bar_a, parity);
      parity ^= 1;
      tc::tc_fence_after();
      // epilogue 1: pool = max over the phase accumulators of this lane
      int mx[16];
#pragma unroll
      for (int e = 0; e < 16; ++e) mx[e] = INT_MIN;
      for (int ph = 0; ph < nph1; ++ph) {
        uint32_t r[16];
        tc::tmem_ld16(tmem + lane_base + ph * 16, r);
        tc::tmem_ld_wait();
#pragma unroll
        for (int e = 0; e < 16; ++e) mx[e] = max(mx[e], (int)r[e]);
      }
      if (p.act1 == LBCNN_ACT_RELU) {
#pragma unroll
        for (int e = 0; e < 16; ++e) mx[e] = max(mx[e], 0);
      }
      if (p.n_layers == 1) {
        if (in_range && b < nb) {
          float* Hrow = p.Hout + ((long long)cand * p.n_img + img0 + b) * p.F;
#pragma unroll
          for (int e = 0; e < 16; ++e)
            if (e < p.Cout1) Hrow[(e * p.Ho1 + i1) * p.Wo1 + j1] = p.scale * (float)mx[e];
        }
      } else if (in_range) {
        // balanced radix-64 digits of the pooled map -> phase plane (i1 % P2, j1 % P2) of layer 2
        uint32_t lo[4] = {0, 0, 0, 0}, hi[4] = {0, 0, 0, 0};
#pragma unroll
        for (int e = 0; e < 16; ++e) {
          const int v = mx[e];
          const int l = ((v + 32) & 63) - 32;
          const int h = (v - l) >> 6;
          lo[e >> 2] |= (uint32_t)(l & 255) << (8 * (e & 3));
          hi[e >> 2] |= (uint32_t)(h & 255) << (8 * (e & 3));
        }
        const int sy = i1 % p.P2, sx = j1 % p.P2;
        const int pos = p.base0 + (b * p.Hq + i1 / p.P2) * p.Wq + j1 / p.P2;
        uint8_t* dst = smem + p.off_pl + (sy * p.P2 + sx) * p.plane_bytes + pos * 16;
        *reinterpret_cast<uint4*>(dst) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
        *reinterpret_cast<uint4*>(dst + p.NPOS2 * 16) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
      }
    }
    if (p.n_layers == 1) continue;
    // ---- layer 2: tiles of 128 positions of the (halo-sharing) pooled output grid ----
    for (int t2 = 0; t2 < p.T2; ++t2) {
      tc::fence_proxy_async();
      tc::tc_fence_before();
      __syncthreads();
      if (tid == 0) {
        tc::tc_fence_after();
        for (int py = 0; py < p.P2; ++py)
          for (int px = 0; px < p.P2; ++px) {
            const uint32_t d = tmem + (py * p.P2 + px) * p.N2;
            uint32_t acc = 0;
            for (int dy = 0; dy < p.k2; ++dy) {
              const int ry = py + dy - p.pd2, qy = floordiv(ry, p.P2), sy = ry - qy * p.P2;
              for (int dx = 0; dx < p.k2; ++dx) {
                const int rx = px + dx - p.pd2, qx = floordiv(rx, p.P2), sx = rx - qx * p.P2;
                const uint32_t a_addr = s_base + p.off_pl + (sy * p.P2 + sx) * p.plane_bytes +
                                        (p.base0 + t2 * 128 + qy * p.Wq + qx) * 16;
                const uint64_t da = tc::smem_desc(a_addr, p.NPOS2 * 16, 128, tc::LAYOUT_NONE);
                const uint64_t db = tc::smem_desc(s_base + p.off_w2 + (dy * p.k2 + dx) * (p.N2 * 32), p.N2 * 16, 128, tc::LAYOUT_NONE);
                tc::mma_i8(d, da, db, idesc2, acc);
                acc = 1;
              }
            }
          }
        tc::mma_commit(bar_a);
      }
      tc::mbar_wait(bar_a, parity);
      parity ^= 1;
      tc::tc_fence_after();
      const int m2 = t2 * 128 + tid;
      const int b = m2 / (p.Hq * p.Wq);
      const int rem = m2 - b * (p.Hq * p.Wq);
      const int i2 = rem / p.Wq, j2 = rem - i2 * p.Wq;
      const bool valid = (m2 < p.NM2) && (b < nb) && (i2 < p.Ho2) && (j2 < p.Wo2);
      float* Hrow = p.Hout + ((long long)cand * p.n_img + img0 + (valid ? b : 0)) * p.F;
      for (int c0 = 0; c0 < p.N2; c0 += 16) {
        int mx[16];
#pragma unroll
        for (int e = 0; e < 16; ++e) mx[e] = INT_MIN;
        for (int ph = 0; ph < p.P2 * p.P2; ++ph) {
          uint32_t r[16];
          tc::tmem_ld16(tmem + lane_base + ph * p.N2 + c0, r);
          tc::tmem_ld_wait();
#pragma unroll
          for (int e = 0; e < 16; ++e) mx[e] = max(mx[e], (int)r[e]);
        }
        if (valid) {
#pragma unroll
          for (int e = 0; e < 16; ++e) {
            const int o = c0 + e;
            if (o < p.Cout2) {
              int v = mx[e];
              if (p.act2 == LBCNN_ACT_RELU) v = max(v, 0);
              Hrow[(o * p.Ho2 + i2) * p.Wo2 + j2] = p.scale * (float)v;     // flatten C,H,W
            }
          }
        }
      }
    }
  }
  tc::tc_fence_before();
  __syncthreads();
  if (warp == 0) { tc::tc_fence_after(); tc::tmem_dealloc(tmem, 256); }
}

}  // namespace

// Is the architecture inside the tensor-core kernel's envelope?  Fills the launch parameters if so.
static bool plan_xtc(const lbcnn_handle_s* h, const ArchShape& s, bool has_bias, XtcParams* q, size_t* smem_bytes) {
  if (has_bias || s.n_layers < 1 || s.n_layers > 2) return false;
  for (int l = 0; l < s.n_layers; ++l) {
    const LayerShape& L = s.L[l];
    if (L.conv_type != LBCNN_CONV_FULL || L.pp != 0 || L.cover != 0 || L.pk != L.ps || L.pk < 1) return false;
    if (L.hin % L.pk != 0 || L.win % L.pk != 0) return false;
  }
  XtcParams p{};
  const LayerShape& A = s.L[0];
  p.H = A.hin; p.W = A.win; p.C = A.cin; p.n_layers = s.n_layers;
  p.k1 = A.k; p.pd1 = (A.k - 1) / 2; p.P1 = A.pk; p.Cout1 = A.cout; p.K1 = A.k * A.k * A.cin;
  p.K1p = (p.K1 + 31) / 32 * 32; p.Ho1 = A.hout; p.Wo1 = A.wout; p.act1 = A.act; p.w1_off = (int)A.w_off;
  if (p.Cout1 > 16 || p.K1p > 128 || p.P1 * p.P1 * 16 > 256) return false;
  int halo = 0;
  if (s.n_layers == 2) {
    const LayerShape& Bq = s.L[1];
    p.k2 = Bq.k; p.pd2 = (Bq.k - 1) / 2; p.P2 = Bq.pk; p.Cout2 = Bq.cout; p.Ho2 = Bq.hout; p.Wo2 = Bq.wout;
    p.act2 = Bq.act; p.w2_off = (int)Bq.w_off;
    p.N2 = (p.Cout2 + 15) / 16 * 16;
    if (p.N2 > 256 || p.P2 * p.P2 * p.N2 > 256) return false;
    if (255LL * p.K1 > 8159) return false;                       // two balanced radix-64 int8 digits
    const int hq = (p.pd2 + p.P2 - 1) / p.P2, qmax = (p.P2 - 1 + p.pd2) / p.P2;
    halo = hq > qmax ? hq : qmax;
    p.Wq = p.Wo2 + halo; p.Hq = p.Ho2 + halo; p.base0 = halo * p.Wq + halo;
  }
  // images per CTA: as many as keep one CTA under ~100 KB of shared memory (two CTAs per SM), at most 8
  const int npx = p.H * p.W * p.C;
  const int limit = 100 * 1024;
  int bestB = 0; XtcParams best{}; size_t best_smem = 0;
  for (int B = 1; B <= 8; ++B) {
    XtcParams t = p;
    t.B = B; t.NP1 = B * p.Ho1 * p.Wo1; t.T1 = (t.NP1 + 127) / 128;
    t.col_slot_bytes = p.P1 * p.P1 * p.K1p * 128;
    int off = 0;
    auto take = [&](int bytes) { int o = off; off += (bytes + 127) / 128 * 128; return o; };
    t.off_img = take(B * npx);
    t.off_w1 = take(16 * p.K1p);
    if (s.n_layers == 2) {
      t.NM2 = B * p.Hq * p.Wq; t.T2 = (t.NM2 + 127) / 128;
      t.NPOS2 = (p.base0 + t.T2 * 128 + halo * p.Wq + halo + 8 + 7) / 8 * 8;
      t.plane_bytes = 2 * t.NPOS2 * 16;
      t.off_w2 = take(p.k2 * p.k2 * p.N2 * 32);
      t.off_pl = take(p.P2 * p.P2 * t.plane_bytes);
      if (t.NPOS2 * 16 >= (1 << 18)) break;
    }
    const int fixed = off;
    // cache the im2col rows of every layer-1 tile across candidates when they fit
    t.cache = (fixed + t.T1 * t.col_slot_bytes <= limit) ? 1 : 0;
    t.off_col = take((t.cache ? t.T1 : 1) * t.col_slot_bytes);
    if (off > limit && B > 1) break;
    if ((size_t)off > (size_t)h->max_smem_optin) break;
    bestB = B; best = t; best_smem = (size_t)off;
  }
  if (!bestB) return false;
  *q = best; *smem_bytes = best_smem;
  return true;
}

bool lb_expand_tc_usable(const lbcnn_handle_s* h, const ArchShape& s, bool has_bias) {
  XtcParams q; size_t sm;
  return plan_xtc(h, s, has_bias, &q, &sm);
}

int lb_launch_expand_tc(lbcnn_handle_s* h, const ArchShape& s, float feature_scale, const uint8_t* d_images, int64_t n,
                        const int8_t* d_kernels, int n_cand, float* d_H, cudaStream_t st) {
  XtcParams p; size_t smem = 0;
  if (!plan_xtc(h, s, false, &p, &smem)) return LBCNN_ERR_INVALID_ARCH;
  LbPhase ph(h, LBCNN_PHASE_EXPAND, st);
  p.img = d_images; p.n_img = n; p.ker = d_kernels; p.n_weights = (int)s.n_weights; p.n_cand = n_cand;
  p.Hout = d_H; p.F = s.F; p.scale = feature_scale;
  const long long batches = (n + p.B - 1) / p.B;
  // candidates per CTA: enough CTAs for ~8 waves of 2 CTAs per SM, otherwise as many candidates as possible
  // per CTA (they share the staged images and, when cached, the im2col rows)
  int cpc = n_cand;
  const long long want = 8LL * 2 * h->n_sm;
  while (cpc > 1 && batches * ((n_cand + cpc - 1) / cpc) < want) cpc = (cpc + 1) / 2;
  p.cand_per_cta = cpc;
  const int gy = (n_cand + cpc - 1) / cpc;
  if (batches > 2147483647LL || gy > 65535) return LBCNN_ERR_INVALID_ARG;
  LB_CUDA_OK(cudaFuncSetAttribute(expand_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  dim3 grid((unsigned)batches, (unsigned)gy);
  expand_tc_kernel<<<grid, 128, smem, st>>>(p);
  h->launches += 1;
  LB_CUDA_OK(cudaGetLastError());
  return LBCNN_OK;
}
