// expand.cu -- K1: the LB-CNN expander: up to three (binary convolution -> optional
// relu -> max-pool) macro-layers, flatten in C,H,W order, one multiply by feature_scale, H written once.
//
// v1 (SIMT, exact int32): one CTA owns one image and a group of candidates.  The image sits in
// shared memory with a zero border (the convolution's zero padding, PAPER.md:53 pad=1), every layer's
// pooled output is written to the next layer's zero-bordered shared buffer, so intermediates never
// touch HBM.  A thread owns one pooled output position for 4 output channels: it evaluates the
// convolution at each in-image cell of the pooling window (padding never wins, cover_all windows are
// clipped to the image) and keeps the running maximum.  Weights (+-1) sit in shared memory as int32
// [tap][Cout padded to 4] so one 128-bit broadcast load feeds four IMADs.
#include "internal.h"

namespace {

struct LayerDev {
  int conv_type, nk, k, act, pk, ps, pp;
  int cin, cout, hin, win, hout, wout;
  int P;          // nk padded to a multiple of 4
  int w_off;      // offset in one candidate's kernel set
  int b_off;      // offset in one candidate's bias set
  int sw_off;     // offset (int32 words) of this layer's weights in the shared weight area
  int sb_off;     // offset of this layer's bias in the shared bias area
  int in_off;     // offset (words) of this layer's zero-bordered input buffer in shared memory
  int out_pad;    // border of the NEXT layer's input buffer (0 for the last layer)
};

struct ExpandParams {
  int n_layers;
  LayerDev L[3];
  int n_cand, cand_per_block;
  int n_weights, n_bias;
  int act_words;    // words of all activation buffers (zeroed once)
  int w_words, b_words;
  long long F;
  long long n;
  long long out_rows;   // rows per candidate of the output buffer (>= n)
  float scale;
  const uint8_t* img;
  const int8_t* ker;
  const int32_t* bias;
  float* H;
};

template <int KS>
__device__ __forceinline__ void run_layer(const LayerDev& L, const int* __restrict__ in, int* __restrict__ out_s,
                                          float* __restrict__ out_g, const int* __restrict__ w,
                                          const int* __restrict__ b, float scale) {
  const int k = KS ? KS : L.k;
  const int pc = (k - 1) / 2;
  const int wp_in = L.win + 2 * pc;
  const int plane_in = (L.hin + 2 * pc) * wp_in;
  const int P4 = L.P >> 2;
  const bool full = (L.conv_type == LBCNN_CONV_FULL);
  const int groups = full ? P4 : L.cin * P4;
  const int n_items = groups * L.hout * L.wout;
  const int wp_out = L.wout + 2 * L.out_pad;
  const int plane_out = (L.hout + 2 * L.out_pad) * wp_out;
  const int4* __restrict__ w4 = reinterpret_cast<const int4*>(w);

  for (int item = threadIdx.x; item < n_items; item += blockDim.x) {
    const int j = item % L.wout;
    const int t = item / L.wout;
    const int i = t % L.hout;
    const int g = t / L.hout;
    int y0 = i * L.ps - L.pp, x0 = j * L.ps - L.pp;
    int y1 = min(y0 + L.pk, L.hin), x1 = min(x0 + L.pk, L.win);
    y0 = max(y0, 0); x0 = max(x0, 0);
    int m0 = INT_MIN, m1 = INT_MIN, m2 = INT_MIN, m3 = INT_MIN;
    int o0;          // first of the 4 output channels of this item
    int nvalid;      // how many of the 4 are real channels
    int c_in = 0, mg = g;
    if (full) { o0 = g * 4; nvalid = min(4, L.cout - o0); }
    else { c_in = g / P4; mg = g % P4; o0 = c_in * L.nk + mg * 4; nvalid = min(4, L.nk - mg * 4); }
    int b0 = 0, b1 = 0, b2 = 0, b3 = 0;
    if (nvalid > 0) b0 = b[o0];
    if (nvalid > 1) b1 = b[o0 + 1];
    if (nvalid > 2) b2 = b[o0 + 2];
    if (nvalid > 3) b3 = b[o0 + 3];
    for (int yy = y0; yy < y1; ++yy)
      for (int xx = x0; xx < x1; ++xx) {
        int a0 = b0, a1 = b1, a2 = b2, a3 = b3;
        // padded coordinates: in-image (yy,xx) sits at (yy+pc, xx+pc); tap (dy,dx) reads (yy+dy, xx+dx)
        const int* ip = in + yy * wp_in + xx;
        if (full) {
          const int4* wq = w4 + mg;
          for (int c = 0; c < L.cin; ++c) {
            const int* ic = ip + c * plane_in;
#pragma unroll
            for (int dy = 0; dy < k; ++dy)
#pragma unroll
              for (int dx = 0; dx < k; ++dx) {
                const int v = ic[dy * wp_in + dx];
                const int4 ww = *wq; wq += P4;
                a0 += v * ww.x; a1 += v * ww.y; a2 += v * ww.z; a3 += v * ww.w;
              }
          }
        } else {
          const int* ic = ip + c_in * plane_in;
          const int4* wq = w4 + (c_in * k * k) * P4 + mg;
#pragma unroll
          for (int dy = 0; dy < k; ++dy)
#pragma unroll
            for (int dx = 0; dx < k; ++dx) {
              const int v = ic[dy * wp_in + dx];
              const int4 ww = *wq; wq += P4;
              a0 += v * ww.x; a1 += v * ww.y; a2 += v * ww.z; a3 += v * ww.w;
            }
        }
        if (L.act == LBCNN_ACT_RELU) { a0 = max(a0, 0); a1 = max(a1, 0); a2 = max(a2, 0); a3 = max(a3, 0); }
        m0 = max(m0, a0); m1 = max(m1, a1); m2 = max(m2, a2); m3 = max(m3, a3);
      }
    const int mm[4] = {m0, m1, m2, m3};
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      if (q < nvalid) {
        const int o = o0 + q;
        if (out_g) out_g[((long long)o * L.hout + i) * L.wout + j] = scale * (float)mm[q];   // flatten C,H,W
        else out_s[o * plane_out + (i + L.out_pad) * wp_out + (j + L.out_pad)] = mm[q];
      }
    }
  }
}

__global__ void __launch_bounds__(256) expand_kernel(const ExpandParams p) {
  extern __shared__ __align__(16) int smem[];
  int* act = smem;                       // activation buffers (image + pooled maps), zero-bordered
  int* sw = smem + p.act_words;          // weights of the current candidate, all layers
  int* sb = sw + p.w_words;              // biases of the current candidate
  const long long img_idx = blockIdx.x;

  for (int t = threadIdx.x; t < p.act_words; t += blockDim.x) act[t] = 0;
  __syncthreads();
  {  // image -> act[L0.in_off] planar [c][h+2p][w+2p]
    const LayerDev& L = p.L[0];
    const int pc = (L.k - 1) / 2;
    const int wp = L.win + 2 * pc, plane = (L.hin + 2 * pc) * wp;
    const int npix = L.hin * L.win * L.cin;
    const uint8_t* src = p.img + img_idx * npix;
    for (int t = threadIdx.x; t < npix; t += blockDim.x) {
      const int c = t % L.cin;
      const int x = (t / L.cin) % L.win;
      const int y = t / (L.cin * L.win);
      act[L.in_off + c * plane + (y + pc) * wp + (x + pc)] = src[t];
    }
  }
  const int k_begin = blockIdx.y * p.cand_per_block;
  const int k_end = min(k_begin + p.cand_per_block, p.n_cand);
  for (int kc = k_begin; kc < k_end; ++kc) {
    __syncthreads();   // previous candidate done with sw/sb (and the image is in place)
    const int8_t* kw = p.ker + (long long)kc * p.n_weights;
    for (int l = 0; l < p.n_layers; ++l) {
      const LayerDev& L = p.L[l];
      const int kk = L.k * L.k;
      const int nw = L.nk * L.cin * kk;
      // source [q][c][dy][dx] (q = o or m)  ->  shared [(c*k+dy)*k+dx][P] + q; padding entries stay 0
      for (int t = threadIdx.x; t < L.cin * kk * L.P; t += blockDim.x) {
        const int q = t % L.P, tap = t / L.P;
        sw[L.sw_off + t] = (q < L.nk) ? (int)kw[L.w_off + q * (L.cin * kk) + tap] : 0;
      }
      (void)nw;
      for (int t = threadIdx.x; t < L.cout; t += blockDim.x)
        sb[L.sb_off + t] = p.bias ? p.bias[(long long)kc * p.n_bias + L.b_off + t] : 0;
    }
    __syncthreads();
    float* Hrow = p.H + ((long long)kc * p.out_rows + img_idx) * p.F;
    for (int l = 0; l < p.n_layers; ++l) {
      const LayerDev& L = p.L[l];
      const bool last = (l == p.n_layers - 1);
      const int* in = act + L.in_off;
      int* out_s = last ? nullptr : act + p.L[l + 1].in_off;
      float* out_g = last ? Hrow : nullptr;
      if (L.k == 3) run_layer<3>(L, in, out_s, out_g, sw + L.sw_off, sb + L.sb_off, p.scale);
      else if (L.k == 5) run_layer<5>(L, in, out_s, out_g, sw + L.sw_off, sb + L.sb_off, p.scale);
      else run_layer<0>(L, in, out_s, out_g, sw + L.sw_off, sb + L.sb_off, p.scale);
      if (!last) __syncthreads();
    }
  }
}

}  // namespace

size_t lb_expand_ws_bytes(const lbcnn_handle_s* h, const ArchShape& s, bool has_bias, int n_cand) {
  return h->force_simt_expand ? 0 : lb_expand_tc_ws_bytes(h, s, has_bias, n_cand);
}

int lb_launch_expand(lbcnn_handle_s* h, const ArchShape& s, float feature_scale, const uint8_t* d_images, int64_t n,
                     const int8_t* d_kernels, const int32_t* d_bias, int n_cand, float* d_H, void* xw, size_t xw_bytes,
                     cudaStream_t st, bool prepared, int64_t out_rows) {
  if (!h->force_simt_expand && lb_expand_tc_usable(h, s, d_bias != nullptr))
    return lb_launch_expand_tc(h, s, feature_scale, d_images, n, d_kernels, n_cand, d_H, xw, xw_bytes, st, prepared, out_rows);
  LbPhase ph(h, LBCNN_PHASE_EXPAND, st);
  ExpandParams p{};
  p.n_layers = s.n_layers;
  int act_words = 0, w_words = 0, b_words = 0, max_items = 0;
  for (int l = 0; l < s.n_layers; ++l) {
    const LayerShape& S = s.L[l];
    LayerDev& L = p.L[l];
    L.conv_type = S.conv_type; L.nk = S.nk; L.k = S.k; L.act = S.act; L.pk = S.pk; L.ps = S.ps; L.pp = S.pp;
    L.cin = S.cin; L.cout = S.cout; L.hin = S.hin; L.win = S.win; L.hout = S.hout; L.wout = S.wout;
    L.P = (S.nk + 3) / 4 * 4;
    L.w_off = (int)S.w_off; L.b_off = (int)S.b_off;
    const int pc = (S.k - 1) / 2;
    L.in_off = act_words;
    act_words += S.cin * (S.hin + 2 * pc) * (S.win + 2 * pc);
    act_words = (act_words + 3) / 4 * 4;
    L.sw_off = w_words;
    w_words += S.cin * S.k * S.k * L.P;
    L.sb_off = b_words;
    b_words += (S.cout + 3) / 4 * 4;
    L.out_pad = (l + 1 < s.n_layers) ? (s.L[l + 1].k - 1) / 2 : 0;
    const int groups = (S.conv_type == LBCNN_CONV_FULL) ? L.P / 4 : S.cin * (L.P / 4);
    const int items = groups * S.hout * S.wout;
    if (items > max_items) max_items = items;
  }
  p.act_words = act_words; p.w_words = w_words; p.b_words = b_words;
  const size_t smem = sizeof(int) * ((size_t)act_words + w_words + b_words);
  if (smem > (size_t)h->max_smem_optin) return LBCNN_ERR_INVALID_ARCH;
  if (s.max_abs >= (1LL << 31)) return LBCNN_ERR_INVALID_ARCH;   // int32 accumulators must stay exact
  p.n_cand = n_cand;
  p.cand_per_block = n_cand < 8 ? n_cand : 8;
  p.n_weights = (int)s.n_weights; p.n_bias = (int)s.n_bias;
  p.F = s.F; p.n = n; p.out_rows = out_rows > 0 ? out_rows : n; p.scale = feature_scale;
  p.img = d_images; p.ker = d_kernels; p.bias = d_bias; p.H = d_H;
  int threads = (max_items + 31) / 32 * 32;
  if (threads < 64) threads = 64;
  if (threads > 256) threads = 256;
  LB_CUDA_OK(cudaFuncSetAttribute(expand_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int gy = (n_cand + p.cand_per_block - 1) / p.cand_per_block;
  // grid.x is limited to 2^31-1 images; grid.y to 65535 candidate groups
  if (n > 2147483647LL || gy > 65535) return LBCNN_ERR_INVALID_ARG;
  dim3 grid((unsigned)n, (unsigned)gy);
  expand_kernel<<<grid, threads, smem, st>>>(p);
  h->launches += 1;
  LB_CUDA_OK(cudaGetLastError());
  return LBCNN_OK;
}
