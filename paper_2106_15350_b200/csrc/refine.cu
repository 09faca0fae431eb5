// refine.cu -- gradient refinement of the output layer on the full training set (the notebook's
// Cell 10: "training the output layer with the full dataset", +0.73 pp on MNIST).  The paper
// names neither loss nor optimiser; reading DESIGN.md R18 (= SPEC.md:324, 355): softmax cross-entropy, adaptive moment
// estimation with the standard constants, mini-batches, binary kernels frozen (the features are an input here).
// Everything in fp64 (weights, moments, logits, gradients) on the DMMA tile engine, so the trajectory follows the
// oracle's to rounding order; W is rounded to fp32 once at the end.  The steps are sequential by nature: five small
// launches per mini-batch (gather, logits, softmax, gradient, Adam).
#include "gemm_launch.cuh"
#include <cmath>

namespace {

__global__ void rf_init_kernel(const float* __restrict__ W, long long n, double* __restrict__ Wd, double* __restrict__ m,
                               double* __restrict__ v, double* __restrict__ loss, int epochs) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t < n) { Wd[t] = (double)W[t]; m[t] = 0.0; v[t] = 0.0; }
  if (t < epochs) loss[t] = 0.0;
}

// sample j of the epoch is (a j + b) mod n
__global__ void rf_gather_kernel(const float* __restrict__ H, long long n, long long F, unsigned long long a, unsigned long long b,
                                 long long j0, int nb, float* __restrict__ Hb) {
  const int r = blockIdx.y;
  const long long f = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= nb || f >= F) return;
  const long long i = (long long)((a * (unsigned long long)(j0 + r) + b) % (unsigned long long)n);
  Hb[(long long)r * F + f] = H[i * F + f];
}

// one warp per row: Z -> P - T (softmax with the row maximum subtracted), loss -= log P[y]
__global__ void __launch_bounds__(256) rf_softmax_kernel(double* __restrict__ Z, int nb, int c, const int32_t* __restrict__ y,
                                                         long long n, unsigned long long a, unsigned long long b, long long j0,
                                                         double* __restrict__ loss) {
  const int r = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (r >= nb) return;
  double* z = Z + (long long)r * c;
  const int lab = y[(long long)((a * (unsigned long long)(j0 + r) + b) % (unsigned long long)n)];
  double mx = -1.0e300;
  for (int j = lane; j < c; j += 32) mx = fmax(mx, z[j]);
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, d));
  double s = 0.0;
  for (int j = lane; j < c; j += 32) s += exp(z[j] - mx);
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
  for (int j = lane; j < c; j += 32) {
    const double p = exp(z[j] - mx) / s;
    if (j == lab) atomicAdd(loss, -log(p));
    z[j] = p - (j == lab ? 1.0 : 0.0);
  }
}

__global__ void rf_adam_kernel(double* __restrict__ W, double* __restrict__ m, double* __restrict__ v, const double* __restrict__ G,
                               long long n, double lr, double b1, double b2, double eps, double c1, double c2) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  const double g = G[t];
  const double mm = b1 * m[t] + (1.0 - b1) * g, vv = b2 * v[t] + (1.0 - b2) * g * g;
  m[t] = mm; v[t] = vv;
  W[t] -= lr * (mm * c1) / (sqrt(vv * c2) + eps);
}

__global__ void rf_finish_kernel(const double* __restrict__ Wd, long long n, float* __restrict__ W, const double* __restrict__ acc,
                                 int epochs, double inv_n, float* __restrict__ loss_out) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t < n) W[t] = (float)Wd[t];
  if (loss_out && t < epochs) loss_out[t] = (float)(acc[t] * inv_n);
}

unsigned long long rf_mix(unsigned long long z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
unsigned long long rf_draw(unsigned long long seed, unsigned long long gen, unsigned long long child, unsigned long long i) {
  const unsigned long long G1 = 0x9E3779B97F4A7C15ull, G2 = 0xBF58476D1CE4E5B9ull;
  const unsigned long long key = rf_mix(seed ^ (G1 * (gen + 1)));
  const unsigned long long ckey = rf_mix(key + G2 * (child + 1));
  return rf_mix(ckey + G1 * (i + 1));
}
unsigned long long rf_gcd(unsigned long long x, unsigned long long y) { while (y) { const unsigned long long t = x % y; x = y; y = t; } return x; }

struct RfLayout { size_t wd, m, v, g, hb, z, loss, total; };
void rf_layout(int64_t F, int c, int batch, int epochs, RfLayout* L) {
  size_t off = 0;
  auto take = [&](int64_t bytes) { size_t o = off; off += (size_t)lb_align_up(bytes, 256); return o; };
  L->wd = take(F * c * 8); L->m = take(F * c * 8); L->v = take(F * c * 8); L->g = take(F * c * 8);
  L->hb = take((int64_t)batch * F * 4); L->z = take((int64_t)batch * c * 8); L->loss = take((int64_t)epochs * 8 + 8);
  L->total = off;
}

}  // namespace

size_t lb_refine_ws_bytes(int64_t F, int n_classes, int batch, int epochs) {
  RfLayout L;
  rf_layout(F, n_classes, batch, epochs, &L);
  return L.total;
}

int lb_launch_refine(lbcnn_handle_s* h, void* ws, const float* d_H, int64_t n, int64_t F, float h_scale, const int32_t* d_labels,
                     int c, const lbcnn_refine_t& cfg, float* d_W, float* d_loss, cudaStream_t st) {
  RfLayout L;
  rf_layout(F, c, cfg.batch, cfg.epochs, &L);
  char* base = reinterpret_cast<char*>(ws);
  double* Wd = reinterpret_cast<double*>(base + L.wd);
  double* m = reinterpret_cast<double*>(base + L.m);
  double* v = reinterpret_cast<double*>(base + L.v);
  double* G = reinterpret_cast<double*>(base + L.g);
  float* Hb = reinterpret_cast<float*>(base + L.hb);
  double* Z = reinterpret_cast<double*>(base + L.z);
  double* loss = reinterpret_cast<double*>(base + L.loss);
  const long long nw = (long long)F * c;
  const unsigned gw = (unsigned)((nw + 255) / 256);
  const double hs = (double)h_scale;
  int rc;
  const unsigned gi = (unsigned)(((nw > cfg.epochs ? nw : cfg.epochs) + 255) / 256);   // also covers loss[0 .. epochs)
  rf_init_kernel<<<gi > 1 ? gi : 1, 256, 0, st>>>(d_W, nw, Wd, m, v, loss, cfg.epochs);
  h->launches += 1;
  long long t = 0;
  for (int e = 0; e < cfg.epochs; ++e) {
    unsigned long long a = 1, b = 0;
    if (n > 1) {
      a = 1 + rf_draw(cfg.seed, (unsigned long long)e, 0, 0) % (unsigned long long)(n - 1);
      while (rf_gcd(a, (unsigned long long)n) != 1) a = a % (unsigned long long)(n - 1) + 1;
      b = rf_draw(cfg.seed, (unsigned long long)e, 0, 1) % (unsigned long long)n;
    }
    for (long long j0 = 0; j0 < n; j0 += cfg.batch) {
      const int nb = (int)((n - j0 < cfg.batch) ? n - j0 : cfg.batch);
      dim3 gg((unsigned)((F + 255) / 256), (unsigned)nb);
      rf_gather_kernel<<<gg, 256, 0, st>>>(d_H, n, F, a, b, j0, nb, Hb);
      {
        GemmP g{};                                                   // Z = hs * Hb W
        g.A = Hb; g.sAr = F; g.sAk = 1; g.bA = 0;
        g.B = Wd; g.sBr = 1; g.sBk = c; g.bB = 0;
        g.C = Z; g.ldc = c; g.bC = 0;
        g.M = nb; g.N = c; g.K = (int)F; g.alpha = hs; g.accumulate = 0; g.lower = 0; g.diag = 0.0;
        rc = launch_gemm<float, double, double, true, false>(h, g, 1, st);
        if (rc) return rc;
      }
      rf_softmax_kernel<<<(nb + 7) / 8, 256, 0, st>>>(Z, nb, c, d_labels, n, a, b, j0, loss + e);
      {
        GemmP g{};                                                   // G = (hs / nb) Hb^T (P - T)
        g.A = Hb; g.sAr = 1; g.sAk = F; g.bA = 0;
        g.B = Z; g.sBr = 1; g.sBk = c; g.bB = 0;
        g.C = G; g.ldc = c; g.bC = 0;
        g.M = (int)F; g.N = c; g.K = nb; g.alpha = hs / (double)nb; g.accumulate = 0; g.lower = 0; g.diag = 0.0;
        rc = launch_gemm<float, double, double, false, false>(h, g, 1, st);
        if (rc) return rc;
      }
      t += 1;
      const double c1 = 1.0 / (1.0 - std::pow((double)cfg.beta1, (double)t)), c2 = 1.0 / (1.0 - std::pow((double)cfg.beta2, (double)t));
      rf_adam_kernel<<<gw > 1 ? gw : 1, 256, 0, st>>>(Wd, m, v, G, nw, (double)cfg.lr, (double)cfg.beta1, (double)cfg.beta2, (double)cfg.eps, c1, c2);
      h->launches += 3;
    }
  }
  const unsigned gf = (unsigned)(((nw > cfg.epochs ? nw : cfg.epochs) + 255) / 256);
  rf_finish_kernel<<<gf > 1 ? gf : 1, 256, 0, st>>>(Wd, nw, d_W, loss, cfg.epochs, 1.0 / (double)n, d_loss);
  h->launches += 1;
  LB_CUDA_OK(cudaGetLastError());
  return LBCNN_OK;
}
