// probe: a PT2 reduction WITHOUT a hash table in HBM, end to end on synthetic records, to see what the round-2 design can reach.
//   stage 1  records {key, H psi, H_aa} are generated in registers (standing in for the enumeration) and partitioned by a
//            CTA-synchronous counting sort into B1 bins, every CTA writing its own segment of each bin (coalesced runs, no atomics
//            on global memory);
//   stage 2  one bin at a time (all CTAs on the same bin, CTA c takes the segment level-1 CTA c wrote): a second counting sort
//            into B2 sub-bins through a scratch that is small enough to stay in L2;
//   stage 3  one sub-bin per CTA pass: gather its per-CTA segments into shared memory, deduplicate there (index hash, fp64
//            shared atomics), add v^2 / (E - H_aa) per distinct key.
// Every key id appears exactly `dup` times, so the number of distinct keys and the sum have closed forms to check against.
// Stand-alone: shares no code with the library.  nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 pipe_bench.cu
#include <cstdio>
#include <cstdlib>
#include <cstdint>
#include <cuda_runtime.h>
typedef unsigned long long u64;
struct __align__(32) Rec { u64 ka, kb; double v, h; };
__device__ __host__ __forceinline__ u64 mix(u64 x) { x += 0x9E3779B97F4A7C15ull; x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull; x = (x ^ (x >> 27)) * 0x94D049BB133111EBull; return x ^ (x >> 31); }
__device__ __forceinline__ void st256(void* p, const Rec& x) { asm volatile("st.global.v4.u64 [%0], {%1,%2,%3,%4};" ::"l"(p), "l"(x.ka), "l"(x.kb), "l"(__double_as_longlong(x.v)), "l"(__double_as_longlong(x.h)) : "memory"); }
__device__ __forceinline__ Rec ld256(const void* p) { u64 a, b, c, d; asm volatile("ld.global.v4.u64 {%0,%1,%2,%3}, [%4];" : "=l"(a), "=l"(b), "=l"(c), "=l"(d) : "l"(p) : "memory"); return Rec{a, b, __longlong_as_double(c), __longlong_as_double(d)}; }
__device__ __forceinline__ Rec ld256cs(const void* p) { u64 a, b, c, d; asm volatile("ld.global.cs.v4.u64 {%0,%1,%2,%3}, [%4];" : "=l"(a), "=l"(b), "=l"(c), "=l"(d) : "l"(p) : "memory"); return Rec{a, b, __longlong_as_double(c), __longlong_as_double(d)}; }
#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { printf("ERR %s line %d\n", cudaGetErrorString(e_), __LINE__); exit(1); } } while (0)

constexpr int kT = 1024;      // threads per partition CTA
constexpr int kN = 2048;      // records per counting-sort round
constexpr int kB = 1024;      // bins per level (B1 = B2)

// bin of a key at a level: 10 bits of a hash of the key
__device__ __forceinline__ int bin_of(u64 ka, int level) { return (int)((mix(ka) >> (level == 1 ? 54 : 44)) & (kB - 1)); }

// One counting-sort round over buf[0..cnt): histogram, scan, scatter into srt, write bin runs to out[bin][cta][segu[bin]..).
// All kT threads call it.  `cap` records per (bin, CTA) segment; records that do not fit are counted in *drop.
__device__ __forceinline__ void sort_round(const Rec* buf, Rec* srt, unsigned short* sbin, unsigned* hist, unsigned* base, unsigned* segu,
                                           unsigned* wtot, int cnt, int level, Rec* out, unsigned cap, u64& drop) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  constexpr int PER = kN / kT;
  unsigned rk[PER]; int bn[PER];
#pragma unroll
  for (int q = 0; q < PER; ++q) {
    const int t = threadIdx.x + q * kT;
    bn[q] = -1;
    if (t < cnt) { bn[q] = bin_of(buf[t].ka, level); rk[q] = atomicAdd(&hist[bn[q]], 1u); }
  }
  __syncthreads();
  {
    unsigned v = hist[threadIdx.x], x = v;                       // kB == kT: one bin per thread
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { unsigned y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
    if (lane == 31) wtot[warp] = x;
    __syncthreads();
    if (warp == 0) { unsigned w = wtot[lane], sx = w; for (int o = 1; o < 32; o <<= 1) { unsigned y = __shfl_up_sync(0xffffffffu, sx, o); if (lane >= o) sx += y; } wtot[lane] = sx - w; }
    __syncthreads();
    base[threadIdx.x] = wtot[warp] + x - v;
  }
  __syncthreads();
#pragma unroll
  for (int q = 0; q < PER; ++q)
    if (bn[q] >= 0) { const unsigned d = base[bn[q]] + rk[q]; srt[d] = buf[threadIdx.x + q * kT]; sbin[d] = (unsigned short)bn[q]; }
  __syncthreads();
#pragma unroll
  for (int q = 0; q < PER; ++q) {
    const int t = threadIdx.x + q * kT;
    if (t < cnt) {
      const int b = sbin[t];
      const unsigned p = segu[b] + ((unsigned)t - base[b]);
      if (p < cap) st256(out + ((u64)b * gridDim.x + blockIdx.x) * cap + p, srt[t]); else ++drop;
    }
  }
  __syncthreads();
  segu[threadIdx.x] += hist[threadIdx.x]; hist[threadIdx.x] = 0;
  __syncthreads();
}

struct PartSmem { Rec* buf; Rec* srt; unsigned* hist; unsigned* base; unsigned* segu; unsigned short* sbin; };
__device__ __forceinline__ PartSmem carve(unsigned char* sm) {
  PartSmem s;
  s.buf = reinterpret_cast<Rec*>(sm); s.srt = s.buf + kN;
  s.hist = reinterpret_cast<unsigned*>(s.srt + kN); s.base = s.hist + kB; s.segu = s.base + kB;
  s.sbin = reinterpret_cast<unsigned short*>(s.segu + kB);
  return s;
}
constexpr size_t kPartSmem = 2 * (size_t)kN * sizeof(Rec) + 3 * (size_t)kB * sizeof(unsigned) + (size_t)kN * sizeof(unsigned short);

// ---------------------------------------------------------------- stage 1: generate + level-1 partition
__global__ void __launch_bounds__(kT, 1)
stage1_kernel(Rec* pool1, unsigned cap1, int rounds, u64 n_keys, unsigned* used1, u64* dropped) {
  extern __shared__ __align__(32) unsigned char sm[];
  PartSmem S = carve(sm);
  __shared__ unsigned wtot[32];
  S.hist[threadIdx.x] = 0; S.segu[threadIdx.x] = 0;
  __syncthreads();
  u64 drop = 0;
  for (int rd = 0; rd < rounds; ++rd) {
#pragma unroll
    for (int q = 0; q < kN / kT; ++q) {
      const u64 g = ((u64)rd * gridDim.x + blockIdx.x) * kN + threadIdx.x + q * kT;
      const u64 id = g % n_keys;
      S.buf[threadIdx.x + q * kT] = Rec{mix(id) | 1ull, mix(id ^ 0xABCDEF0123ull), 1.0, -2.0 - (double)(id & 15)};
    }
    __syncthreads();
    sort_round(S.buf, S.srt, S.sbin, S.hist, S.base, S.segu, wtot, kN, 1, pool1, cap1, drop);
  }
  used1[(size_t)threadIdx.x * gridDim.x + blockIdx.x] = min(S.segu[threadIdx.x], cap1);
  if (drop) atomicAdd(dropped, drop);
}

// ---------------------------------------------------------------- stage 2: level-2 partition of bin b through the scratch
__global__ void __launch_bounds__(kT, 1)
stage2_kernel(const Rec* __restrict__ pool1, const unsigned* __restrict__ used1, unsigned cap1, int b, Rec* scratch, unsigned cap2,
              unsigned* used2, u64* dropped) {
  extern __shared__ __align__(32) unsigned char sm[];
  PartSmem S = carve(sm);
  __shared__ unsigned wtot[32];
  S.hist[threadIdx.x] = 0; S.segu[threadIdx.x] = 0;
  __syncthreads();
  const unsigned n = used1[(size_t)b * gridDim.x + blockIdx.x];
  const Rec* src = pool1 + ((u64)b * gridDim.x + blockIdx.x) * cap1;
  u64 drop = 0;
  for (unsigned off = 0; off < n; off += kN) {
    const int cnt = (int)min((unsigned)kN, n - off);
#pragma unroll
    for (int q = 0; q < kN / kT; ++q) { const int t = threadIdx.x + q * kT; if (t < cnt) S.buf[t] = ld256cs(src + off + t); }
    __syncthreads();
    sort_round(S.buf, S.srt, S.sbin, S.hist, S.base, S.segu, wtot, cnt, 2, scratch, cap2, drop);
  }
  used2[(size_t)threadIdx.x * gridDim.x + blockIdx.x] = min(S.segu[threadIdx.x], cap2);
  if (drop) atomicAdd(dropped, drop);
}

// ---------------------------------------------------------------- stage 3: gather a sub-bin, dedupe in shared memory, reduce
constexpr int kT3 = 512, kM = 3072;
__global__ void __launch_bounds__(kT3)
stage3_kernel(const Rec* __restrict__ scratch, const unsigned* __restrict__ used2, unsigned cap2, int P, double e_s, double* out /* [2]: sum, distinct */,
              u64* dropped) {
  extern __shared__ __align__(32) unsigned char sm[];
  Rec* rec = reinterpret_cast<Rec*>(sm);                          // [kM]
  int* tab = reinterpret_cast<int*>(rec + kM);                   // [2 kM]
  __shared__ unsigned off[kT3 + 1];
  __shared__ double wsum[2][kT3 / 32];
  double acc = 0.0, cnt = 0.0;
  for (int s = blockIdx.x; s < kB; s += gridDim.x) {
    for (int t = threadIdx.x; t < 2 * kM; t += kT3) tab[t] = -1;
    // exclusive scan of the P segment lengths of sub-bin s (P <= kT3), serial over warps: P is small
    if (threadIdx.x < P) off[threadIdx.x + 1] = used2[(size_t)s * P + threadIdx.x];
    if (threadIdx.x == 0) off[0] = 0;
    __syncthreads();
    if (threadIdx.x == 0) for (int c = 0; c < P; ++c) off[c + 1] += off[c];
    __syncthreads();
    const int m = min((int)off[P], kM);
    if (threadIdx.x == 0 && (int)off[P] > kM) atomicAdd(dropped, (u64)(off[P] - kM));
    for (int t = threadIdx.x; t < m; t += kT3) {
      int lo = 0, hi = P;                                        // segment c with off[c] <= t < off[c + 1]
      while (hi - lo > 1) { const int md = (lo + hi) >> 1; if (off[md] <= (unsigned)t) lo = md; else hi = md; }
      rec[t] = ld256(scratch + ((u64)s * P + lo) * cap2 + (t - off[lo]));
    }
    __syncthreads();
    for (int t = threadIdx.x; t < m; t += kT3) {
      const u64 ka = rec[t].ka, kb = rec[t].kb;
      unsigned h = (unsigned)(mix(ka ^ (kb * 0x9E3779B97F4A7C15ull)) >> 20) % (2 * kM);
      for (;;) {
        const int cur = atomicCAS(&tab[h], -1, t);
        if (cur == -1) break;
        if (rec[cur].ka == ka && rec[cur].kb == kb) { atomicAdd(&rec[cur].v, rec[t].v); rec[t].h = __longlong_as_double(0x7ff8000000000001ll); break; }
        if (++h == 2 * kM) h = 0;
      }
    }
    __syncthreads();
    for (int t = threadIdx.x; t < m; t += kT3) {
      const double hh = rec[t].h;
      if (hh == hh) { const double v = rec[t].v; acc += v * v / (e_s - hh); cnt += 1.0; }
    }
    __syncthreads();
  }
  for (int o = 16; o > 0; o >>= 1) { acc += __shfl_xor_sync(0xffffffffu, acc, o); cnt += __shfl_xor_sync(0xffffffffu, cnt, o); }
  if ((threadIdx.x & 31) == 0) { wsum[0][threadIdx.x >> 5] = acc; wsum[1][threadIdx.x >> 5] = cnt; }
  __syncthreads();
  if (threadIdx.x == 0) { double a = 0, c = 0; for (int w = 0; w < kT3 / 32; ++w) { a += wsum[0][w]; c += wsum[1][w]; } atomicAdd(out, a); atomicAdd(out + 1, c); }
}

int main(int argc, char** argv) {
  const int log2_total = argc > 1 ? atoi(argv[1]) : 31;          // records
  const int dup = argc > 2 ? atoi(argv[2]) : 2;
  cudaDeviceProp prop; CK(cudaGetDeviceProperties(&prop, 0));
  const int P = prop.multiProcessorCount;
  const int rounds = (int)(((1ull << log2_total) / ((u64)P * kN)));
  const u64 total = (u64)rounds * P * kN, n_keys = total / dup;
  const u64 total_used = n_keys * dup;                            // ids 0..n_keys-1 appear dup times; the remainder once more
  const double per_seg1 = (double)total / kB / P, per_seg2 = per_seg1 / kB;
  const unsigned cap1 = (unsigned)(per_seg1 + 8.0 * sqrt(per_seg1) + 64.0), cap2 = (unsigned)(per_seg2 + 6.0 * sqrt(per_seg2) + 8.0);
  printf("%s, %d SMs; %llu records (%.1f GB), %llu keys x %d; level-1 segment %.0f records (cap %u), level-2 segment %.1f (cap %u), scratch %.0f MB\n",
         prop.name, P, total, total * 32 / 1e9, n_keys, dup, per_seg1, cap1, per_seg2, cap2, (double)kB * P * cap2 * 32 / 1048576.0);
  Rec *pool1, *scratch; unsigned *used1, *used2; u64* dropped; double* out;
  CK(cudaMalloc(&pool1, (size_t)kB * P * cap1 * sizeof(Rec)));
  CK(cudaMalloc(&scratch, (size_t)kB * P * cap2 * sizeof(Rec)));
  CK(cudaMalloc(&used1, (size_t)kB * P * 4)); CK(cudaMalloc(&used2, (size_t)kB * P * 4));
  CK(cudaMalloc(&dropped, 8)); CK(cudaMalloc(&out, 16));
  CK(cudaMemset(dropped, 0, 8)); CK(cudaMemset(out, 0, 16));
  const size_t smem3 = (size_t)kM * sizeof(Rec) + 2 * (size_t)kM * sizeof(int);
  CK(cudaFuncSetAttribute(stage1_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kPartSmem));
  CK(cudaFuncSetAttribute(stage2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kPartSmem));
  CK(cudaFuncSetAttribute(stage3_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem3));
  int per_sm3 = 0; CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm3, stage3_kernel, kT3, smem3));
  cudaEvent_t e0, e1, e2; cudaEventCreate(&e0); cudaEventCreate(&e1); cudaEventCreate(&e2);
  const double e_s = 1.0;
  cudaEventRecord(e0);
  stage1_kernel<<<P, kT, kPartSmem>>>(pool1, cap1, rounds, n_keys, used1, dropped);
  cudaEventRecord(e1);
  for (int b = 0; b < kB; ++b) {
    stage2_kernel<<<P, kT, kPartSmem>>>(pool1, used1, cap1, b, scratch, cap2, used2, dropped);
    stage3_kernel<<<P * per_sm3, kT3, smem3>>>(scratch, used2, cap2, P, e_s, out, dropped);
  }
  cudaEventRecord(e2); CK(cudaEventSynchronize(e2)); CK(cudaGetLastError());
  float ms1, ms23; cudaEventElapsedTime(&ms1, e0, e1); cudaEventElapsedTime(&ms23, e1, e2);
  double h[2]; u64 d = 0;
  CK(cudaMemcpy(h, out, 16, cudaMemcpyDeviceToHost)); CK(cudaMemcpy(&d, dropped, 8, cudaMemcpyDeviceToHost));
  double expect = 0.0;                                            // sum over ids of count^2 / (e_s + 2 + (id & 15))
  const u64 extra = total - total_used;                           // ids < extra appear dup + 1 times
  for (int r = 0; r < 16; ++r) {
    const u64 n_r = n_keys / 16 + ((u64)r < n_keys % 16 ? 1 : 0); // ids with id & 15 == r
    const u64 x_r = extra / 16 + ((u64)r < extra % 16 ? 1 : 0);   // of those, the ones below `extra`
    expect += ((double)(n_r - x_r) * dup * dup + (double)x_r * (dup + 1) * (dup + 1)) / (e_s + 2.0 + r);
  }
  printf("stage 1 (generate + partition into %d bins): %8.1f ms  %6.2f G rec/s\n", kB, ms1, total / (ms1 * 1e6));
  printf("stages 2+3 (%d x [partition into %d sub-bins, dedupe + reduce], %d launches): %8.1f ms  %6.2f G rec/s\n", kB, kB, 2 * kB, ms23, total / (ms23 * 1e6));
  printf("whole pipeline: %8.1f ms  %6.2f G rec/s;  dropped %llu;  distinct %.0f (expected %llu);  sum %.9e (expected %.9e, rel %.2e)\n",
         ms1 + ms23, total / ((ms1 + ms23) * 1e6), d, h[1], n_keys, h[0], expect, fabs(h[0] - expect) / expect);
  return 0;
}
