// noalloc.cu -- ONE entry point that allocates nothing: the energy reduction E = sum_i E_i of K8 (eq. 2
// takes F = -grad E of this total; the workspace path does it inside k_force_out, force.cu,
// with its block partials in a cudaMalloc'ed array of the workspace).
//
// Why: some callers cannot call cudaMalloc -- code under CUDA graph capture, tight serving loops, harnesses that forbid
// it -- and creating a workspace allocates.  nnp_energy_sum_static needs no workspace: its scratch (the per-block partial
// sums and the ticket of the "last block adds the partials in index order" reduction) is a file-scope
// `static __device__` array of a fixed, modest size, which every GPU that loads the library holds until exit
// (NNP_STATIC_MAX_ATOMS / 256 doubles + one 256-byte line for the ticket = 33 024 bytes).
//
// The array's name is a host-side stand-in in host code, not a device address: the entry point resolves it once per
// device, with that device current, through cudaGetSymbolAddress, and hands the address to the kernel.
//
// Shared state: every call (of every thread and stream, on one device) uses the SAME array.  The ticket must be zero
// when a kernel starts: it is cleared on the stream before every launch (and the last block leaves it zero).  Two calls
// whose kernels overlap on the GPU (different streams, no dependency between them) race on the partials and the ticket
// and give wrong sums: callers serialise them (one stream, or events).  Calls in one stream are ordered and safe.
#include <cuda_runtime.h>
#include <cstdint>
#include <mutex>
#include "../../include/nnp.h"

namespace {

constexpr int NA_THREADS = 256;
constexpr int NA_MAX_BLOCKS = NNP_STATIC_MAX_ATOMS / NA_THREADS;   // 4096
constexpr int NA_HEAD = 256 / sizeof(double);                       // first 256 bytes: the ticket (one 32-bit word used)
constexpr int NA_MAX_DEVICES = 64;

// [0, NA_HEAD): ticket line;  [NA_HEAD, NA_HEAD + NA_MAX_BLOCKS): fp64 block partials
static __device__ __align__(256) double g_esum_scratch[NA_HEAD + NA_MAX_BLOCKS];

// Same reduction as k_force_out (force.cu): fp64 block partials by a shuffle tree, then the last block to take the ticket
// adds the partials in index order (lane-strided, shuffle tree) -- no floating-point atomics, bitwise reproducible.
__global__ void __launch_bounds__(NA_THREADS)
k_energy_sum_static(const float* __restrict__ e_atom, int n, double e_scale, double* __restrict__ scratch,
                    double* __restrict__ energy) {
  __shared__ double wsum[NA_THREADS / 32];
  __shared__ bool last;
  unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch);
  double* epart = scratch + NA_HEAD;
  const int i = blockIdx.x * NA_THREADS + threadIdx.x;
  const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5;
  double e = (i < n) ? (double)e_atom[i] : 0.0;
  for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
  if (lane == 0) wsum[wp] = e;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int k = 0; k < NA_THREADS / 32; ++k) t += wsum[k];
    epart[blockIdx.x] = t;
    __threadfence();
    last = (atomicAdd(ticket, 1u) == gridDim.x - 1);
  }
  __syncthreads();
  if (!last || wp != 0) return;
  __threadfence();
  double t = 0.0;
  for (int k = lane; k < (int)gridDim.x; k += 32) t += __ldcg(epart + k);
  for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
  if (lane == 0) { *energy = t * e_scale; *ticket = 0u; }
}

// device address of the scratch array, resolved once per device (with that device current)
std::mutex g_mu;
double* g_scratch_ptr[NA_MAX_DEVICES] = {};

int scratch_of_current_device(double** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= NA_MAX_DEVICES) { cudaGetLastError(); return NNP_ERR_CUDA; }
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_ptr[dev]) {
    double* p = nullptr;
    if (cudaGetSymbolAddress((void**)&p, g_esum_scratch) != cudaSuccess || !p) { cudaGetLastError(); return NNP_ERR_CUDA; }
    g_scratch_ptr[dev] = p;
  }
  *out = g_scratch_ptr[dev];
  return NNP_OK;
}

}  // namespace

extern "C" int nnp_energy_sum_static(void* cuda_stream, int64_t n, const float* d_e_atom, double e_scale,
                                     double* d_energy) {
  if (n < 0 || !d_energy || (n > 0 && !d_e_atom)) return NNP_ERR_INVALID_ARG;
  if (n > NNP_STATIC_MAX_ATOMS) return NNP_ERR_STATIC_LIMIT;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  double* scratch = nullptr;
  const int rc = scratch_of_current_device(&scratch);
  if (rc != NNP_OK) return rc;
  if (n == 0) {
    if (cudaMemsetAsync(d_energy, 0, sizeof(double), st) != cudaSuccess) { cudaGetLastError(); return NNP_ERR_CUDA; }
    return NNP_OK;
  }
  // the ticket starts at zero whatever an earlier (possibly aborted) call left behind
  if (cudaMemsetAsync(scratch, 0, 256, st) != cudaSuccess) { cudaGetLastError(); return NNP_ERR_CUDA; }
  const unsigned nb = (unsigned)((n + NA_THREADS - 1) / NA_THREADS);
  k_energy_sum_static<<<nb, NA_THREADS, 0, st>>>(d_e_atom, (int)n, e_scale, scratch, d_energy);
  if (cudaGetLastError() != cudaSuccess) return NNP_ERR_CUDA;
  return NNP_OK;
}
