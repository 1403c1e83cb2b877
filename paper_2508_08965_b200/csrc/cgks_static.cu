// cgks_static.cu -- cgks_compute_dt_static (include/cgks.h): the CFL time step of a bare array of cell averages for callers
// that have no device memory to give the library and may not ask the CUDA allocator for any.
//
// Every other entry point works on a context whose buffers live in a workspace the caller allocated (cgks_create), and
// cgks_compute_dt keeps its running minimum in that workspace.  Some callers cannot produce a workspace at all: a run
// monitor or in-situ hook that is handed one Q array inside a job whose framework allocator (PyTorch's caching allocator,
// say) already owns all of HBM, so that a raw cudaMalloc fails; or a time loop that must not stall, where cudaMalloc /
// cudaFree are off limits because they synchronise the whole device.  For them the reduction's scratch memory is the
// file-scope array below.  It is part of the library image: each GPU that loads libcgks.so holds these 33 kB until the
// process exits, whether or not the entry point is ever called.
//
// This file is self-contained on purpose (own kernels, own error string): nothing in cgks_api.cu changes because of it.
#include "../../include/cgks.h"

#include <cuda_runtime.h>
#include <math.h>
#include <mutex>
#include <string>

namespace {

constexpr int ST_TPB = 256;                                  // threads per block
constexpr int ST_CHUNK = 4096;                               // cells per block: 16 per thread, fixed -> the partials (and so
                                                             // the result) do not depend on the device's SM count
constexpr int ST_MAX_BLOCKS = CGKS_STATIC_MAX_CELLS / ST_CHUNK;   // 4096
constexpr int ST_HEAD = 32;                                  // doubles in front of the partials (256 B): word 0 = bad-cell flag
constexpr int ST_MAX_DEVICES = 64;

// [0, ST_HEAD): header, must be ZERO when the first kernel starts (cleared by every call); [ST_HEAD, ...): one partial
// minimum per block, fully overwritten by every call before it is read (stale contents of the last call are harmless).
// In HOST code this name is only a handle for cudaGetSymbolAddress -- it is not a device address and must never be handed
// to a kernel; scratch_of_current_device() below resolves it.
static __device__ __align__(256) double g_static_scratch[ST_HEAD + ST_MAX_BLOCKS];

thread_local std::string g_static_err;
std::mutex g_static_mu;
double* g_static_ptr[ST_MAX_DEVICES] = {};                   // device address of g_static_scratch, per device ordinal

int fail(int code, const std::string& msg) { g_static_err = msg; return code; }

// Set-up, once per device, with that device current: the device address of the scratch array.  Allocates nothing (the
// array came with the module); on the very first call it may make the CUDA runtime load the module.
cudaError_t scratch_of_current_device(double** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  const bool cached = dev >= 0 && dev < ST_MAX_DEVICES;
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (cached && g_static_ptr[dev]) { *out = g_static_ptr[dev]; return cudaSuccess; }
  double* p = nullptr;
  e = cudaGetSymbolAddress((void**)&p, g_static_scratch);
  if (e != cudaSuccess) return e;
  if (!p) return cudaErrorInvalidSymbol;
  if (cached) g_static_ptr[dev] = p;
  *out = p;
  return cudaSuccess;
}

struct StaticCfl { double gamma, mu_ref, omega, T_ref, cfl, h[3]; };

// Variant of cfl_kernel (kernels_setup.cuh, reading S3) for a uniform Cartesian mesh and cell
// averages in the USER layout Q [5][n]: block b reduces cells [b * ST_CHUNK, (b + 1) * ST_CHUNK) to partial[b].
__global__ void __launch_bounds__(ST_TPB) cfl_static_partial_kernel(long n, const double* __restrict__ Q, StaticCfl p,
                                                                    double* __restrict__ scratch) {
  double dtmin = INFINITY;
  bool bad = false;
  const long c0 = (long)blockIdx.x * ST_CHUNK;
  const long c1 = (c0 + ST_CHUNK < n) ? c0 + ST_CHUNK : n;
  for (long c = c0 + threadIdx.x; c < c1; c += ST_TPB) {
    const double rho = Q[c], mx = Q[n + c], my = Q[2 * n + c], mz = Q[3 * n + c], E = Q[4 * n + c];
    const double U[3] = { mx / rho, my / rho, mz / rho };
    const double pr = (p.gamma - 1.0) * (E - 0.5 * rho * (U[0] * U[0] + U[1] * U[1] + U[2] * U[2]));
    if (!(rho > 0.0) || !(pr > 0.0)) { bad = true; continue; }
    const double cs = sqrt(p.gamma * pr / rho);
    double rate = 0.0, hmin = INFINITY;
#pragma unroll
    for (int ax = 0; ax < 3; ax++) { rate += (fabs(U[ax]) + cs) / p.h[ax]; hmin = fmin(hmin, p.h[ax]); }
    dtmin = fmin(dtmin, p.cfl / rate);
    if (p.mu_ref > 0.0) {
      double mu = p.mu_ref;
      if (p.omega != 0.0) mu *= pow((pr / rho) / p.T_ref, p.omega);
      dtmin = fmin(dtmin, p.cfl * hmin * hmin / (3.0 * mu / rho));
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) dtmin = fmin(dtmin, __shfl_xor_sync(0xffffffffu, dtmin, o));
  __shared__ double sm[ST_TPB / 32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0) sm[wid] = dtmin;
  __syncthreads();
  if (wid == 0) {
    dtmin = (lane < ST_TPB / 32) ? sm[lane] : INFINITY;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dtmin = fmin(dtmin, __shfl_xor_sync(0xffffffffu, dtmin, o));
    if (lane == 0) scratch[ST_HEAD + blockIdx.x] = dtmin;
  }
  if (bad) atomicOr((int*)scratch, 1);
}

// One block: minimum of the nb partials -> d_dt[0]; the bad-cell flag -> d_bad[0] (if wanted).
__global__ void __launch_bounds__(ST_TPB) cfl_static_final_kernel(int nb, const double* __restrict__ scratch,
                                                                  double* __restrict__ d_dt, int* __restrict__ d_bad) {
  double dtmin = INFINITY;
  for (int b = threadIdx.x; b < nb; b += ST_TPB) dtmin = fmin(dtmin, scratch[ST_HEAD + b]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) dtmin = fmin(dtmin, __shfl_xor_sync(0xffffffffu, dtmin, o));
  __shared__ double sm[ST_TPB / 32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0) sm[wid] = dtmin;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < ST_TPB / 32; w++) dtmin = fmin(dtmin, sm[w]);
    d_dt[0] = dtmin;
    if (d_bad) d_bad[0] = *(const int*)scratch;
  }
}

}  // namespace

extern "C" const char* cgks_static_last_error(void) { return g_static_err.c_str(); }

extern "C" int cgks_compute_dt_static(int ni, int nj, int nk, const double* d_Q, const double* h_host,
                                      const cgks_params* params, double cfl, double* d_dt, int* d_bad, void* cuda_stream) {
  if (ni < 1 || nj < 1 || nk < 1) return fail(CGKS_EINVAL, "cgks_compute_dt_static: ni, nj, nk must be positive");
  const double cells = (double)ni * (double)nj * (double)nk;
  if (cells > (double)CGKS_STATIC_MAX_CELLS)
    return fail(CGKS_EINVAL, "cgks_compute_dt_static: " + std::to_string((long long)cells) + " cells exceed the " +
                                 std::to_string((long long)CGKS_STATIC_MAX_CELLS) +
                                 " cells (256^3) the built-in scratch array is sized for; use cgks_compute_dt on a context");
  if (!d_Q || !h_host || !params || !d_dt) return fail(CGKS_EINVAL, "cgks_compute_dt_static: null argument");
  if (!(cfl > 0.0) || !(h_host[0] > 0.0) || !(h_host[1] > 0.0) || !(h_host[2] > 0.0) || !(params->gamma > 1.0) || !(params->T_ref > 0.0))
    return fail(CGKS_EINVAL, "cgks_compute_dt_static: cfl, the three cell sizes and T_ref must be positive and gamma > 1");
  const long n = (long)ni * nj * nk;
  const int nb = (int)((n + ST_CHUNK - 1) / ST_CHUNK);
  cudaStream_t st = (cudaStream_t)cuda_stream;

  double* scratch = nullptr;                                  // DEVICE address of g_static_scratch on the current device
  cudaError_t e = scratch_of_current_device(&scratch);
  if (e != cudaSuccess) return fail(CGKS_ECUDA, std::string("cgks_compute_dt_static: cudaGetSymbolAddress: ") + cudaGetErrorString(e));

  StaticCfl p{ params->gamma, params->mu_ref, params->visc_omega, params->T_ref, cfl, { h_host[0], h_host[1], h_host[2] } };
  // the header keeps whatever the last call left (a raised flag, if that call saw a bad cell): clear it on the stream
  e = cudaMemsetAsync(scratch, 0, ST_HEAD * sizeof(double), st);
  if (e != cudaSuccess) return fail(CGKS_ECUDA, std::string("cgks_compute_dt_static: cudaMemsetAsync: ") + cudaGetErrorString(e));
  cfl_static_partial_kernel<<<nb, ST_TPB, 0, st>>>(n, d_Q, p, scratch);
  cfl_static_final_kernel<<<1, ST_TPB, 0, st>>>(nb, scratch, d_dt, d_bad);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(CGKS_ECUDA, std::string("cgks_compute_dt_static: launch: ") + cudaGetErrorString(e));
  g_static_err.clear();
  return CGKS_OK;
}
