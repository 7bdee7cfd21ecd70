// tree_energy_static (include/tree.h "entry point that allocates nothing"): the energy sums of tree_energy for callers
// that must not call cudaMalloc (stream capture, tight serving loops, harnesses that forbid it).  The scratch the existing
// path keeps in a cudaMalloc'ed DevInfo (energy_kernel's two FP64 accumulators, bh_force.cu) lives here in ONE file-scope
// device array of fixed size, which every GPU that loads the library holds until the process exits.
//
// In host code the array's name is a host-side stand-in, not a device address: the address a kernel may use comes from
// cudaGetSymbolAddress, asked once per device with that device current (static_scratch below).
#include <cuda_runtime.h>
#include <cstdio>
#include <mutex>

#include "../../include/tree.h"

namespace {

constexpr int ES_THREADS = 256;
constexpr int ES_CHUNK = 4096;         // particles per block (16 per thread)
constexpr int ES_MAX_BLOCKS = 32768;   // partial sums the scratch holds
static_assert((long long)ES_MAX_BLOCKS * ES_CHUNK == TREE_ENERGY_STATIC_MAX_N, "tree.h states the limit");
constexpr int ES_HEAD = 256;           // bytes in front of the partial sums: the arrival counter
constexpr size_t ES_BYTES = ES_HEAD + (size_t)ES_MAX_BLOCKS * sizeof(double2);  // 512.25 KiB
constexpr int ES_MAX_DEVICES = 64;

// layout: [0, 4) arrival counter (must be 0 when a launch starts) | [256, 256 + 16 n_blocks) per-block (kinetic, potential)
static __device__ __align__(256) unsigned char g_energy_scratch[ES_BYTES];

thread_local char tl_err[256] = "";

int fail(int code, const char *what, cudaError_t ce = cudaSuccess) {
  if (ce != cudaSuccess) snprintf(tl_err, sizeof tl_err, "tree_energy_static: %s: %s", what, cudaGetErrorString(ce));
  else snprintf(tl_err, sizeof tl_err, "tree_energy_static: %s", what);
  return code;
}

// Device address of g_energy_scratch on `device`, which must be the current device.  Asked once per device.
std::mutex g_mu;
void *g_scratch_addr[ES_MAX_DEVICES] = {};

cudaError_t static_scratch(int device, void **out) {
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_addr[device]) {
    void *p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_energy_scratch);
    if (e != cudaSuccess) return e;
    g_scratch_addr[device] = p;
  }
  *out = g_scratch_addr[device];
  return cudaSuccess;
}

// Block b sums particles [4096 b, 4096 (b + 1)) in FP64 from the FP32 inputs (the terms of energy_kernel, bh_force.cu),
// writes its pair of sums to part[b] and takes an arrival ticket; the block that arrives last adds the partial sums in
// index order and writes out[0] = kinetic, out[1] = potential: the result does not depend on the order in which blocks ran.
__global__ void __launch_bounds__(ES_THREADS) energy_static_kernel(const float *__restrict__ mass, const float *__restrict__ vel,
                                                                   const float *__restrict__ pot, long long N,
                                                                   unsigned *count, double2 *part, double *__restrict__ out) {
  __shared__ double s_k[ES_THREADS], s_p[ES_THREADS];
  __shared__ bool s_last;
  const int tid = threadIdx.x;
  const long long base = blockIdx.x * (long long)ES_CHUNK;
  double ke = 0.0, pe = 0.0;
#pragma unroll 4
  for (int k = 0; k < ES_CHUNK / ES_THREADS; ++k) {
    const long long i = base + k * ES_THREADS + tid;
    if (i < N) {
      const double m = (double)mass[i];
      if (vel) {
        const float vx = vel[3 * i], vy = vel[3 * i + 1], vz = vel[3 * i + 2];
        ke += 0.5 * m * ((double)vx * vx + (double)vy * vy + (double)vz * vz);
      }
      if (pot) pe += 0.5 * m * (double)pot[i];
    }
  }
  s_k[tid] = ke; s_p[tid] = pe;
  __syncthreads();
  for (int w = ES_THREADS / 2; w > 0; w >>= 1) {
    if (tid < w) { s_k[tid] += s_k[tid + w]; s_p[tid] += s_p[tid + w]; }
    __syncthreads();
  }
  if (tid == 0) {
    part[blockIdx.x] = make_double2(s_k[0], s_p[0]);
    __threadfence();
    s_last = atomicAdd(count, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  ke = 0.0; pe = 0.0;
  for (unsigned b = tid; b < gridDim.x; b += ES_THREADS) {
    const double2 v = __ldcg(&part[b]);
    ke += v.x; pe += v.y;
  }
  s_k[tid] = ke; s_p[tid] = pe;
  __syncthreads();
  for (int w = ES_THREADS / 2; w > 0; w >>= 1) {
    if (tid < w) { s_k[tid] += s_k[tid + w]; s_p[tid] += s_p[tid + w]; }
    __syncthreads();
  }
  if (tid == 0) {
    out[0] = s_k[0];
    out[1] = s_p[0];
    *count = 0;  // the next call on this device finds the counter at zero
  }
}

}  // namespace

extern "C" int tree_energy_static(int device, void *cuda_stream, const float *mass, const float *vel, const float *pot,
                                  long long N, double *out) {
  tl_err[0] = 0;
  if (device < 0 || device >= ES_MAX_DEVICES) return fail(TREE_ERR_ARG, "device out of range");
  if (N < 0) return fail(TREE_ERR_ARG, "N < 0");
  if (N > TREE_ENERGY_STATIC_MAX_N) {
    snprintf(tl_err, sizeof tl_err,
             "tree_energy_static: N = %lld exceeds TREE_ENERGY_STATIC_MAX_N = %lld (the static scratch holds %d partial sums "
             "of %d particles each); use tree_energy", N, (long long)TREE_ENERGY_STATIC_MAX_N, ES_MAX_BLOCKS, ES_CHUNK);
    return TREE_ERR_ARG;
  }
  if (N > 0 && (!mass || !out)) return fail(TREE_ERR_ARG, "mass or out is NULL");
  int prev = -1;
  cudaError_t e = cudaGetDevice(&prev);
  if (e != cudaSuccess) return fail(TREE_ERR_CUDA, "cudaGetDevice", e);
  if (prev != device && (e = cudaSetDevice(device)) != cudaSuccess) return fail(TREE_ERR_CUDA, "cudaSetDevice", e);
  int rc = TREE_OK;
  void *scratch = nullptr;
  if ((e = static_scratch(device, &scratch)) != cudaSuccess) {
    rc = fail(TREE_ERR_CUDA, "cudaGetSymbolAddress", e);
  } else if (N > 0) {
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    unsigned *count = (unsigned *)scratch;
    double2 *part = (double2 *)((unsigned char *)scratch + ES_HEAD);
    const unsigned blocks = (unsigned)((N + ES_CHUNK - 1) / ES_CHUNK);
    // the counter must start at zero; a kernel that ran to its end has reset it, one that was aborted has not
    if ((e = cudaMemsetAsync(count, 0, sizeof(unsigned), stream)) != cudaSuccess) {
      rc = fail(TREE_ERR_CUDA, "cudaMemsetAsync", e);
    } else {
      energy_static_kernel<<<blocks, ES_THREADS, 0, stream>>>(mass, vel, pot, N, count, part, out);
      if ((e = cudaGetLastError()) != cudaSuccess) rc = fail(TREE_ERR_CUDA, "energy_static_kernel", e);
    }
  }
  if (prev != device) cudaSetDevice(prev);
  return rc;
}

extern "C" const char *tree_energy_static_error(void) { return tl_err; }
