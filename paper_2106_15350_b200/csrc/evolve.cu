// evolve.cu -- a non-random candidate generator on top of the search driver: one generation of an
// elitist genetic search over binary kernel sets.  The paper names "nature inspired optimization methods (such as
// genetic algorithms or swarm intelligence methods)" as the step beyond random kernels without
// giving an algorithm; this follows reading DESIGN.md R17 (include/lbcnn.h states it in full).  Everything is integer /
// byte work and the random numbers are a counter-based splitmix64 finaliser keyed by (seed, generation, child, draw), so
// the result is bit-exact against the oracle, which implements the same generator on its own.
#include "internal.h"
#include <mutex>

namespace {

constexpr unsigned long long G1 = 0x9E3779B97F4A7C15ull, G2 = 0xBF58476D1CE4E5B9ull, G3 = 0x94D049BB133111EBull;

__host__ __device__ __forceinline__ unsigned long long mix64(unsigned long long z) {
  z = (z ^ (z >> 30)) * G2;
  z = (z ^ (z >> 27)) * G3;
  return z ^ (z >> 31);
}

// a NaN accuracy compares with nothing: ranked as minus infinity (R17) so that the ranks stay a permutation
__device__ __forceinline__ float ga_key(float a) { return (a != a) ? __int_as_float(0xff800000) : a; }

// rank by accuracy, best first, equal accuracies by index: order[rank] = candidate, rank_of[candidate] = rank
__global__ void __launch_bounds__(256) ga_rank_kernel(const float* __restrict__ acc, int K, int32_t* __restrict__ order,
                                                      int32_t* __restrict__ rank_of) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= K) return;
  const float ai = ga_key(acc[i]);
  int r = 0;
  for (int j = 0; j < K; ++j) {
    const float aj = ga_key(acc[j]);
    r += (aj > ai || (aj == ai && j < i)) ? 1 : 0;
  }
  order[r] = i;
  rank_of[i] = r;
}

__global__ void __launch_bounds__(256) ga_child_kernel(const int8_t* __restrict__ ker, int K, long long nw, int n_elite,
                                                       unsigned int mut_ppm, unsigned long long key,
                                                       const int32_t* __restrict__ order, const int32_t* __restrict__ rank_of,
                                                       int8_t* __restrict__ next) {
  const int j = blockIdx.y;
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nw) return;
  int8_t* dst = next + (long long)j * nw;
  if (j < n_elite) { dst[t] = ker[(long long)order[j] * nw + t]; return; }
  const unsigned long long ckey = mix64(key + G2 * (unsigned long long)(j + 1));
  int c[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) c[i] = (int)(mix64(ckey + G1 * (unsigned long long)(i + 1)) % (unsigned long long)K);
  const int p1 = (rank_of[c[0]] <= rank_of[c[1]]) ? c[0] : c[1];
  const int p2 = (rank_of[c[2]] <= rank_of[c[3]]) ? c[2] : c[3];
  const unsigned long long d = mix64(ckey + G1 * (unsigned long long)(4 + t + 1));
  int v = ((d & 1ull) == 0ull) ? ker[(long long)p1 * nw + t] : ker[(long long)p2 * nw + t];
  if (((d >> 20) % 1000000ull) < (unsigned long long)mut_ppm) v = -v;
  dst[t] = (int8_t)v;
}

}  // namespace

int lb_launch_evolve(lbcnn_handle_s* h, void* ws, const int8_t* d_kernels, const float* d_acc, int n_cand, int64_t n_weights,
                     int n_elite, uint32_t mut_ppm, uint64_t seed, uint32_t generation, int8_t* d_next, cudaStream_t st) {
  int32_t* order = reinterpret_cast<int32_t*>(ws);
  int32_t* rank_of = order + n_cand;
  ga_rank_kernel<<<(n_cand + 255) / 256, 256, 0, st>>>(d_acc, n_cand, order, rank_of);
  const unsigned long long key = mix64((unsigned long long)seed ^ (G1 * (unsigned long long)(generation + 1)));
  dim3 grid((unsigned)((n_weights + 255) / 256), (unsigned)n_cand);
  ga_child_kernel<<<grid, 256, 0, st>>>(d_kernels, n_cand, n_weights, n_elite, mut_ppm, key, order, rank_of, d_next);
  h->launches += 2;
  LB_CUDA_OK(cudaGetLastError());
  return LBCNN_OK;
}

// ---- lbcnn_evolve_candidates_static: the same generation step without a caller workspace ---------------------------------
// For callers that have no device allocator to draw a workspace from (include/lbcnn.h says who they are).  The ranking
// scratch -- order[n_cand] then rank_of[n_cand], int32 each -- sits in an array that is part of the library image instead.
// 2 * 16384 * 4 B = 128 KB on every GPU that loads liblbcnn, from module load to process exit.
static __device__ __align__(256) int32_t g_evolve_scratch[2 * LBCNN_EVOLVE_STATIC_MAX_CAND];

namespace {

// On the host, `g_evolve_scratch` names a shadow object the runtime uses as a look-up key; it is NOT the device address, and a
// kernel handed &g_evolve_scratch[0] from host code would fault (or scribble on host memory where the GPU can reach it).
// The real address differs per device and comes from cudaGetSymbolAddress with that device current; it is looked up on
// the first call per device and kept here.
constexpr int LB_MAX_DEVICES = 64;
std::mutex g_scratch_mu;
int32_t* g_scratch_addr[LB_MAX_DEVICES];   // zero-initialised: not looked up yet

// scratch address on the calling thread's current device, which must be `device`
int evolve_static_scratch(int device, int32_t** out) {
  if (device < 0 || device >= LB_MAX_DEVICES) return LBCNN_ERR_INVALID_ARG;
  int cur = -1;
  LB_CUDA_OK(cudaGetDevice(&cur));
  if (cur != device) return LBCNN_ERR_INVALID_ARG;
  std::lock_guard<std::mutex> lock(g_scratch_mu);
  if (!g_scratch_addr[device]) {
    void* p = nullptr;
    LB_CUDA_OK(cudaGetSymbolAddress(&p, g_evolve_scratch));   // may load the module on this device: first call = set-up
    if (!p) return LBCNN_ERR_CUDA;
    g_scratch_addr[device] = static_cast<int32_t*>(p);
  }
  *out = g_scratch_addr[device];
  return LBCNN_OK;
}

}  // namespace

extern "C" int lbcnn_evolve_candidates_static(lbcnn_handle_t h, const int8_t* d_kernels, const float* d_acc, int32_t n_cand,
                                              int64_t n_weights, int32_t n_elite, uint32_t mut_ppm, uint64_t seed,
                                              uint32_t generation, int8_t* d_next, void* stream) {
  if (!h || !d_kernels || !d_acc || !d_next || n_cand < 1 || n_weights < 1) return LBCNN_ERR_INVALID_ARG;
  if (n_cand > LBCNN_EVOLVE_STATIC_MAX_CAND) return LBCNN_ERR_STATIC_LIMIT;   // the array is a fixed size: refuse, never spill
  if (n_elite < 0 || n_elite > n_cand || mut_ppm > 1000000u || d_next == d_kernels) return LBCNN_ERR_INVALID_ARG;
  int32_t* scratch = nullptr;
  const int rc = evolve_static_scratch(h->device, &scratch);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  // The array still holds whatever the previous call (any handle, any stream) left in it.  The rank kernel overwrites
  // order[0 .. n_cand) and rank_of[0 .. n_cand) completely (the ranks are a permutation); the clear is there so that this
  // call's result can never depend on the array's history, whatever a later change to the kernels does.
  LB_CUDA_OK(cudaMemsetAsync(scratch, 0, (size_t)n_cand * 8, st));
  return lb_launch_evolve(h, scratch, d_kernels, d_acc, n_cand, n_weights, n_elite, mut_ppm, seed, generation, d_next, st);
}
