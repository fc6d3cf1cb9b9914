// detham_energy_static: the energy step (Eq. 11) for callers that may not allocate - code under CUDA graph
// capture, serving loops, harnesses that forbid cudaMalloc.  Same arithmetic per row as energy.cu's spmv_energy_kernel; the
// partial sums live in a file-scope device array instead of a buffer of the context, so the call needs no context and calls no
// cudaMalloc / cudaFree / allocating library routine.  The array is held by every GPU that loads the library until exit.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include <mutex>

#include "detham.h"

namespace {

constexpr int kRowsPerPart = 1024;  // rows whose partial sums share one entry of the scratch
constexpr int kMaxParts = DETHAM_ENERGY_STATIC_MAX_ROWS / kRowsPerPart;
constexpr int kMaxDevices = 64;
static_assert(DETHAM_ENERGY_STATIC_MAX_ROWS % kRowsPerPart == 0, "the row limit is a whole number of parts");

// {psi^T H psi, psi^T psi} of every part: 8192 x 16 B = 128 KB.  Shared by every call on the device; entry p is written by the
// call's partial kernel before its reduce kernel reads it, so nothing has to start at zero and nothing is cleared.
static __device__ __align__(256) double g_energy_scratch[2 * kMaxParts];

// Device address of the array per device.  In host code the name g_energy_scratch is a host-side stand-in, not a device
// address: only cudaGetSymbolAddress, with the device current, yields the pointer a kernel may be given.
double* g_scratch_ptr[kMaxDevices];
std::mutex g_mu;

thread_local char t_err[256] = "";

// one CTA per part of kRowsPerPart rows, TPR threads per row; the CTA's sums go to part[2 * blockIdx.x ..]
template <int TPR>
__global__ void __launch_bounds__(256)
energy_static_kernel(const int64_t* __restrict__ row_ptr, const int* __restrict__ col, const double* __restrict__ val,
                     const double* __restrict__ psi, int64_t nd, double* __restrict__ y_out, double* __restrict__ part) {
  const int sub = threadIdx.x % TPR;
  constexpr int kRowsPerIter = 256 / TPR;
  const int64_t first = (int64_t)blockIdx.x * kRowsPerPart;
  double num = 0.0, den = 0.0;
  for (int r0 = 0; r0 < kRowsPerPart; r0 += kRowsPerIter) {  // CTA-uniform bounds: the sub-warp shuffles stay convergent
    const int64_t row = first + r0 + threadIdx.x / TPR;
    const bool live = row < nd;
    const int64_t b = live ? row_ptr[row] : 0, e = live ? row_ptr[row + 1] : 0;
    double acc = 0.0;
    for (int64_t k = b + sub; k < e; k += TPR) acc = fma(val[k], __ldg(psi + col[k]), acc);
#pragma unroll
    for (int o = TPR / 2; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o, TPR);
    if (sub == 0 && live) {
      const double p = psi[row];
      if (y_out) y_out[row] = acc;
      num = fma(p, acc, num);
      den = fma(p, p, den);
    }
  }
  __shared__ double sn[8], sd[8];
  for (int o = 16; o > 0; o >>= 1) { num += __shfl_xor_sync(0xffffffffu, num, o); den += __shfl_xor_sync(0xffffffffu, den, o); }
  if ((threadIdx.x & 31) == 0) { sn[threadIdx.x >> 5] = num; sd[threadIdx.x >> 5] = den; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0.0, b = 0.0;
    for (int w = 0; w < 8; ++w) { a += sn[w]; b += sd[w]; }
    part[2 * blockIdx.x] = a;
    part[2 * blockIdx.x + 1] = b;
  }
}

// out = {sum of the parts' psi^T H psi, sum of psi^T psi, their quotient E_S}, in a fixed order
__global__ void energy_static_reduce_kernel(const double* __restrict__ part, int nparts, double* __restrict__ out) {
  __shared__ double sa[256], sb[256];
  double a = 0.0, b = 0.0;
  for (int t = threadIdx.x; t < nparts; t += 256) { a += part[2 * t]; b += part[2 * t + 1]; }
  sa[threadIdx.x] = a; sb[threadIdx.x] = b;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if (threadIdx.x < s) { sa[threadIdx.x] += sa[threadIdx.x + s]; sb[threadIdx.x] += sb[threadIdx.x + s]; }
    __syncthreads();
  }
  if (threadIdx.x == 0) { out[0] = sa[0]; out[1] = sb[0]; out[2] = sa[0] / sb[0]; }
}

dh_status fail(dh_status st, const char* what, cudaError_t e = cudaSuccess) {
  if (e != cudaSuccess) snprintf(t_err, sizeof t_err, "%s: %s", what, cudaGetErrorString(e));
  else snprintf(t_err, sizeof t_err, "%s", what);
  return st;
}

}  // namespace

extern "C" const char* detham_energy_static_error(void) { return t_err; }

extern "C" dh_status detham_energy_static(const int64_t* row_ptr, const int32_t* col, const double* val, const double* psi,
                                          int64_t n_dets, int64_t nnz, double* y_out, double* out3, void* stream) {
  t_err[0] = 0;
  if (!row_ptr || !col || !val || !psi || !out3) return fail(DH_EINVAL, "detham_energy_static: NULL row_ptr, col, val, psi or out3");
  if (n_dets < 1 || nnz < 0) return fail(DH_EINVAL, "detham_energy_static: n_dets must be >= 1 and nnz >= 0");
  if (n_dets > (int64_t)DETHAM_ENERGY_STATIC_MAX_ROWS) {
    snprintf(t_err, sizeof t_err, "detham_energy_static: n_dets = %lld exceeds DETHAM_ENERGY_STATIC_MAX_ROWS = %d (use detham_energy)",
             (long long)n_dets, (int)DETHAM_ENERGY_STATIC_MAX_ROWS);
    return DH_EINVAL;
  }
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(DH_ECUDA, "detham_energy_static: cudaGetDevice", e);
  if (dev < 0 || dev >= kMaxDevices) return fail(DH_EINVAL, "detham_energy_static: device ordinal out of range");
  double* part = nullptr;
  {  // set-up, once per device, with that device current
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_ptr[dev]) {
      void* p = nullptr;
      e = cudaGetSymbolAddress(&p, g_energy_scratch);
      if (e != cudaSuccess || !p) return fail(DH_ECUDA, "detham_energy_static: cudaGetSymbolAddress", e);
      g_scratch_ptr[dev] = static_cast<double*>(p);
    }
    part = g_scratch_ptr[dev];
  }
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const int nparts = (int)((n_dets + kRowsPerPart - 1) / kRowsPerPart);
  const double avg = (double)nnz / (double)n_dets;
  if (avg <= 6) energy_static_kernel<4><<<nparts, 256, 0, s>>>(row_ptr, col, val, psi, n_dets, y_out, part);
  else if (avg <= 24) energy_static_kernel<8><<<nparts, 256, 0, s>>>(row_ptr, col, val, psi, n_dets, y_out, part);
  else energy_static_kernel<32><<<nparts, 256, 0, s>>>(row_ptr, col, val, psi, n_dets, y_out, part);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(DH_ECUDA, "detham_energy_static: launch of the partial kernel", e);
  energy_static_reduce_kernel<<<1, 256, 0, s>>>(part, nparts, out3);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(DH_ECUDA, "detham_energy_static: launch of the reduce kernel", e);
  return DH_OK;
}
