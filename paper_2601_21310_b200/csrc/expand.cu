// Sorting of the deduplicated externals of expand mode (row f2) by their 128-bit key: two stable LSD radix-sort passes
// (low word, then high word) over (word, index) pairs with CUB, then one gather.  A library sort is used here on purpose:
// this is the "next" row's post-processing, not the hot path.
#include <cub/device/device_radix_sort.cuh>

#include "common.cuh"

namespace {

__global__ void iota_kernel(unsigned* idx, int64_t m) {
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < m; t += (int64_t)gridDim.x * blockDim.x) idx[t] = (unsigned)t;
}
__global__ void pick_word_kernel(const u64* __restrict__ keys, const unsigned* __restrict__ idx, int word, int64_t m, u64* __restrict__ out) {
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < m; t += (int64_t)gridDim.x * blockDim.x)
    out[t] = keys[2 * (int64_t)idx[t] + word];
}
__global__ void gather_kernel(const u64* __restrict__ keys, const double* __restrict__ v, const double* __restrict__ score,
                              const unsigned* __restrict__ idx, int64_t m, u64* __restrict__ keys_out, double* __restrict__ v_out,
                              double* __restrict__ score_out) {
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < m; t += (int64_t)gridDim.x * blockDim.x) {
    const int64_t s = idx[t];
    keys_out[2 * t] = keys[2 * s]; keys_out[2 * t + 1] = keys[2 * s + 1];
    if (v_out) v_out[t] = v[s];
    if (score_out) score_out[t] = score[s];
  }
}

}  // namespace

dh_status dh_sort_externals(detham_ctx* c, u64* keys_tmp, double* v_tmp, double* score_tmp, int64_t m, u64* keys_out, double* v_out,
                            double* score_out) {
  if (m >= (1ll << 32)) return DH_EINVAL;
  const int grid = c->sm_count * 8;
  u64 *w0 = nullptr, *w1 = nullptr; unsigned *i0 = nullptr, *i1 = nullptr; void* tmp = nullptr;
  auto cleanup = [&]() { cudaFree(w0); cudaFree(w1); cudaFree(i0); cudaFree(i1); cudaFree(tmp); };
  auto body = [&]() -> dh_status {
    DH_CUDA(c, cudaMalloc(&w0, m * sizeof(u64)));
    DH_CUDA(c, cudaMalloc(&w1, m * sizeof(u64)));
    DH_CUDA(c, cudaMalloc(&i0, m * sizeof(unsigned)));
    DH_CUDA(c, cudaMalloc(&i1, m * sizeof(unsigned)));
    size_t tmp_bytes = 0;
    DH_CUDA(c, cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, w0, w1, i0, i1, m, 0, 64, c->stream));
    DH_CUDA(c, cudaMalloc(&tmp, tmp_bytes));
    iota_kernel<<<grid, 256, 0, c->stream>>>(i0, m);
    for (int word = 1; word >= 0; --word) {  // beta (low) word first, alpha (high) word last: order = (alpha, beta)
      pick_word_kernel<<<grid, 256, 0, c->stream>>>(keys_tmp, i0, word, m, w0);
      DH_CUDA(c, cudaGetLastError());
      DH_CUDA(c, cub::DeviceRadixSort::SortPairs(tmp, tmp_bytes, w0, w1, i0, i1, m, 0, 64, c->stream));
      unsigned* t = i0; i0 = i1; i1 = t;
    }
    gather_kernel<<<grid, 256, 0, c->stream>>>(keys_tmp, v_tmp, score_tmp, i0, m, keys_out, v_out, score_out);
    DH_CUDA(c, cudaGetLastError());
    DH_CUDA(c, cudaStreamSynchronize(c->stream));
    return DH_OK;
  };
  dh_status st = body();
  cleanup();
  return st;
}
