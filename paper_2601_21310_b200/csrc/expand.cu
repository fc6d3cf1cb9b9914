// Sorting of the deduplicated externals of expand mode (row f2) by their 128-bit key: a stable LSD radix sort of (word, index)
// pairs, 8 bits per pass, over the beta word and then the alpha word (only the n_orb bits that can be set), then one gather.
// Per pass: digit histogram per tile of 4096 elements, an exclusive scan of every digit's row of tile counts (one CTA per digit) and
// of the 256 digit totals, stable scatter.  Own kernels: no
// library sort on this row.
#include "common.cuh"

namespace {

constexpr int kSortThreads = 1024;  // 32 warps
constexpr int kSortRounds = 4;      // elements per thread, taken in rounds of 1024 consecutive elements
constexpr int kSortTile = kSortThreads * kSortRounds;

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

// hist[digit * ntiles + tile] = number of elements of the tile with that digit
__global__ void __launch_bounds__(kSortThreads)
radix_hist_kernel(const u64* __restrict__ w, int64_t m, int shift, unsigned* __restrict__ hist, int ntiles) {
  __shared__ unsigned s_hist[256];
  if (threadIdx.x < 256) s_hist[threadIdx.x] = 0;
  __syncthreads();
  const int64_t base = (int64_t)blockIdx.x * kSortTile;
#pragma unroll
  for (int r = 0; r < kSortRounds; ++r) {
    const int64_t e = base + r * kSortThreads + threadIdx.x;
    if (e < m) atomicAdd(&s_hist[(unsigned)(w[e] >> shift) & 255u], 1u);
  }
  __syncthreads();
  if (threadIdx.x < 256) hist[(int64_t)threadIdx.x * ntiles + blockIdx.x] = s_hist[threadIdx.x];
}

// CTA d scans row d of hist (the tiles' counts of digit d) in place, exclusive, and leaves the row's total in totals[d]
__global__ void __launch_bounds__(1024)
radix_rowscan_kernel(unsigned* __restrict__ hist, int ntiles, unsigned* __restrict__ totals) {
  __shared__ unsigned s_warp[32];
  __shared__ unsigned s_carry;
  unsigned* row = hist + (int64_t)blockIdx.x * ntiles;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) s_carry = 0;
  __syncthreads();
  for (int base = 0; base < ntiles; base += 1024) {
    const int t = base + threadIdx.x;
    const unsigned x = t < ntiles ? row[t] : 0u;
    unsigned inc = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const unsigned y = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += y; }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    if (warp == 0) {
      unsigned w = s_warp[lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const unsigned y = __shfl_up_sync(0xffffffffu, w, o); if (lane >= o) w += y; }
      s_warp[lane] = w;  // inclusive over the warps
    }
    __syncthreads();
    const unsigned carry = s_carry;
    const unsigned before = carry + (warp ? s_warp[warp - 1] : 0u) + inc - x;
    if (t < ntiles) row[t] = before;
    __syncthreads();
    if (threadIdx.x == 1023) s_carry = carry + s_warp[31];
    __syncthreads();
  }
  if (threadIdx.x == 0) totals[blockIdx.x] = s_carry;
}

// exclusive scan of the 256 digit totals: where each digit's elements start
__global__ void radix_base_kernel(const unsigned* __restrict__ totals, unsigned* __restrict__ base) {
  __shared__ unsigned s[256];
  s[threadIdx.x] = totals[threadIdx.x];
  __syncthreads();
  if (threadIdx.x == 0) { unsigned run = 0; for (int d = 0; d < 256; ++d) { const unsigned c = s[d]; s[d] = run; run += c; } }
  __syncthreads();
  base[threadIdx.x] = s[threadIdx.x];
}

// stable scatter of one tile: an element goes to (start of its digit for this tile) + (elements of the tile with the same digit
// before it).  Rounds of 1024 consecutive elements; inside a round the order is (warp, lane).
__global__ void __launch_bounds__(kSortThreads)
radix_scatter_kernel(const u64* __restrict__ w_in, const unsigned* __restrict__ i_in, int64_t m, int shift,
                     const unsigned* __restrict__ offs, const unsigned* __restrict__ dbase, int ntiles, u64* __restrict__ w_out,
                     unsigned* __restrict__ i_out) {
  __shared__ unsigned short s_cnt[32][256];
  __shared__ unsigned s_base[256], s_tot[256];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned lt = (1u << lane) - 1u;
  if (threadIdx.x < 256) s_base[threadIdx.x] = dbase[threadIdx.x] + offs[(int64_t)threadIdx.x * ntiles + blockIdx.x];
  const int64_t base = (int64_t)blockIdx.x * kSortTile;
  for (int r = 0; r < kSortRounds; ++r) {
    for (int k = threadIdx.x; k < 32 * 256 / 2; k += kSortThreads) reinterpret_cast<unsigned*>(&s_cnt[0][0])[k] = 0u;
    __syncthreads();
    const int64_t e = base + r * kSortThreads + threadIdx.x;
    const bool valid = e < m;
    const u64 key = valid ? w_in[e] : 0ull;
    const unsigned idx = valid ? i_in[e] : 0u;
    const unsigned d = (unsigned)(key >> shift) & 255u;
    const unsigned peers = __match_any_sync(0xffffffffu, valid ? d : 256u);
    const unsigned rank = __popc(peers & lt);
    if (valid && rank == 0) s_cnt[warp][d] = (unsigned short)__popc(peers);
    __syncthreads();
    if (threadIdx.x < 256) {  // exclusive prefix over the warps, per digit
      unsigned run = 0;
      for (int q = 0; q < 32; ++q) { const unsigned c = s_cnt[q][threadIdx.x]; s_cnt[q][threadIdx.x] = (unsigned short)run; run += c; }
      s_tot[threadIdx.x] = run;
    }
    __syncthreads();
    if (valid) {
      const int64_t pos = (int64_t)s_base[d] + s_cnt[warp][d] + rank;
      DH_CHECK(pos >= 0 && pos < m);
      w_out[pos] = key;
      i_out[pos] = idx;
    }
    __syncthreads();
    if (threadIdx.x < 256) s_base[threadIdx.x] += s_tot[threadIdx.x];
  }
}

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

}  // namespace

// bytes of work space dh_sort_externals needs for m elements
size_t dh_sort_work_bytes(int64_t m) {
  const int64_t ntiles = (m + kSortTile - 1) / kSortTile;
  return 2 * align256((size_t)m * sizeof(u64)) + 2 * align256((size_t)m * sizeof(unsigned)) + align256((size_t)256 * ntiles * sizeof(unsigned)) + 2 * align256(256 * sizeof(unsigned)) + 256;
}

// keys_tmp [m][2], v_tmp, score_tmp (unsorted, may be NULL) -> keys_out, v_out, score_out sorted by (alpha, beta); `work`: device
// buffer of dh_sort_work_bytes(m) bytes
dh_status dh_sort_externals(detham_ctx* c, u64* keys_tmp, double* v_tmp, double* score_tmp, int64_t m, u64* keys_out, double* v_out,
                            double* score_out, void* work) {
  if (m >= (1ll << 32)) return DH_EINVAL;
  const int grid = c->sm_count * 8;
  const int ntiles = (int)((m + kSortTile - 1) / kSortTile);
  char* p = static_cast<char*>(work);
  u64* w0 = reinterpret_cast<u64*>(p); p += align256((size_t)m * sizeof(u64));
  u64* w1 = reinterpret_cast<u64*>(p); p += align256((size_t)m * sizeof(u64));
  unsigned* i0 = reinterpret_cast<unsigned*>(p); p += align256((size_t)m * sizeof(unsigned));
  unsigned* i1 = reinterpret_cast<unsigned*>(p); p += align256((size_t)m * sizeof(unsigned));
  unsigned* hist = reinterpret_cast<unsigned*>(p); p += align256((size_t)256 * ntiles * sizeof(unsigned));
  unsigned* totals = reinterpret_cast<unsigned*>(p); p += align256(256 * sizeof(unsigned));
  unsigned* dbase = reinterpret_cast<unsigned*>(p);
  iota_kernel<<<grid, 256, 0, c->stream>>>(i0, m);
  for (int word = 1; word >= 0; --word) {  // beta (low) word first, alpha (high) word last: order = (alpha, beta)
    pick_word_kernel<<<grid, 256, 0, c->stream>>>(keys_tmp, i0, word, m, w0);
    DH_CUDA(c, cudaGetLastError());
    for (int shift = 0; shift < c->n; shift += 8) {  // bits at or above n_orb are zero in every key
      radix_hist_kernel<<<ntiles, kSortThreads, 0, c->stream>>>(w0, m, shift, hist, ntiles);
      radix_rowscan_kernel<<<256, 1024, 0, c->stream>>>(hist, ntiles, totals);
      radix_base_kernel<<<1, 256, 0, c->stream>>>(totals, dbase);
      radix_scatter_kernel<<<ntiles, kSortThreads, 0, c->stream>>>(w0, i0, m, shift, hist, dbase, ntiles, w1, i1);
      DH_CUDA(c, cudaGetLastError());
      u64* tw = w0; w0 = w1; w1 = tw;
      unsigned* ti = i0; i0 = i1; i1 = ti;
    }
  }
  gather_kernel<<<grid, 256, 0, c->stream>>>(keys_tmp, v_tmp, score_tmp, i0, m, keys_out, v_out, score_out);
  DH_CUDA(c, cudaGetLastError());
  DH_CUDA(c, cudaStreamSynchronize(c->stream));
  return DH_OK;
}
