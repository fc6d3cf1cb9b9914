// probe: the three building blocks a binned PT2 (no random HBM traffic) would be made of, each timed alone:
//   A  shared-memory-staged radix partition: records are generated in registers, staged per bin in shared memory and
//      flushed as full lines with one global atomic per LINE (lock-free ticket scheme, no CTA barrier);
//   B  deduplication of one small bin entirely in shared memory (hash of record indices, fp64 atomics in shared memory);
//   C  merge of records that arrive ORDERED BY TABLE REGION into a big HBM hash table (L2-local probes, no barrier).
// Stand-alone: shares no code with the library.  nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 bin_bench.cu
#include <cstdio>
#include <cstdlib>
#include <cstdint>
#include <cuda_runtime.h>
typedef unsigned long long u64;
struct __align__(32) Rec { u64 ka, kb; double v, h; };
__device__ __forceinline__ u64 mix(u64 x) { x += 0x9E3779B97F4A7C15ull; x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull; x = (x ^ (x >> 27)) * 0x94D049BB133111EBull; return x ^ (x >> 31); }
__device__ __forceinline__ void st256(void* p, u64 a, u64 b, u64 c, u64 d) { asm volatile("st.global.cs.v4.u64 [%0], {%1,%2,%3,%4};" ::"l"(p), "l"(a), "l"(b), "l"(c), "l"(d) : "memory"); }
__device__ __forceinline__ void ld256(const void* p, u64& a, u64& b, u64& c, u64& d) { asm volatile("ld.relaxed.gpu.global.v4.u64 {%0,%1,%2,%3}, [%4];" : "=l"(a), "=l"(b), "=l"(c), "=l"(d) : "l"(p) : "memory"); }
__device__ __forceinline__ void ld256cs(const void* p, u64& a, u64& b, u64& c, u64& d) { asm volatile("ld.global.cs.v4.u64 {%0,%1,%2,%3}, [%4];" : "=l"(a), "=l"(b), "=l"(c), "=l"(d) : "l"(p) : "memory"); }
__device__ __forceinline__ void cas128(void* addr, u64 va, u64 vb, u64& oa, u64& ob) {
  asm volatile("{\n\t.reg .b128 c, v, o;\n\tmov.b128 c, {%2, %3};\n\tmov.b128 v, {%4, %5};\n\tatom.relaxed.gpu.global.cas.b128 o, [%6], c, v;\n\tmov.b128 {%0, %1}, o;\n\t}"
               : "=l"(oa), "=l"(ob) : "l"(0ull), "l"(0ull), "l"(va), "l"(vb), "l"(addr) : "memory");
}
#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { printf("ERR %s line %d\n", cudaGetErrorString(e_), __LINE__); exit(1); } } while (0)

// ------------------------------------------------------------------ A: staged partition
// K records per line, two lines per bin.  tick[b]: tickets handed out; a ticket t writes slot t % K of line (t / K) & 1 in that
// line's use number (t / K) >> 1, once lgen[b][line] says the previous use has been flushed; the LAST writer to finish a line
// (done[b][line] == K - 1) flushes it to the bin's next global line and releases it.
template <int K>
__global__ void __launch_bounds__(1024, 1)
part_kernel(Rec* pool, u64* gcur, int B, u64 cap_lines, int iters, u64 seed, u64* dropped) {
  extern __shared__ __align__(32) unsigned char sm[];
  Rec* stage = reinterpret_cast<Rec*>(sm);                       // [B][2][K]
  unsigned* tick = reinterpret_cast<unsigned*>(stage + (size_t)B * 2 * K);
  unsigned* done = tick + B;                                     // [B][2]
  volatile unsigned* lgen = done + 2 * B;                        // [B][2]
  for (int t = threadIdx.x; t < 5 * B; t += blockDim.x) tick[t] = 0;
  __syncthreads();
  const u64 tid = (u64)blockIdx.x * blockDim.x + threadIdx.x;
  u64 drop = 0;
  for (int it = 0; it < iters; ++it) {
    const u64 r = mix(seed + tid * 1315423911ull + (u64)it * 0x100000001B3ull);
    const int b = (int)(((r >> 32) * (u64)B) >> 32);
    const unsigned t = atomicAdd(&tick[b], 1u);
    const unsigned g = t / K, pos = t % K, line = g & 1u, use = g >> 1;
    Rec* ln = stage + ((size_t)b * 2 + line) * K;
    bool pending = true;
    while (pending) {
      if (lgen[2 * b + line] == use) {
        ln[pos] = Rec{r | 1ull, r * 3ull, 1.0, 2.0};
        __threadfence_block();
        const unsigned d = atomicAdd(&done[2 * b + line], 1u);
        if (d == K - 1) {
          __threadfence_block();
          done[2 * b + line] = 0;
          const u64 gl = atomicAdd(&gcur[b], 1ull);
          if (gl < cap_lines) {
            Rec* dst = pool + ((u64)b * cap_lines + gl) * K;
#pragma unroll
            for (int k = 0; k < K; ++k) { const Rec x = ln[k]; st256(dst + k, x.ka, x.kb, __double_as_longlong(x.v), __double_as_longlong(x.h)); }
          } else drop += K;
          __threadfence_block();
          lgen[2 * b + line] = use + 1;
        }
        pending = false;
      }
    }
  }
  if (drop) atomicAdd(dropped, drop);
}
// A2: the same staging, but every CTA owns a private segment of each bin, so a line's position comes from a shared-memory
// counter and no global atomic sits between two uses of a staging line; NL lines per bin (ring).
template <int K, int NL>
__global__ void __launch_bounds__(1024, 1)
part_private_kernel(Rec* pool, int B, u64 cap_lines /* per (bin, CTA) */, int iters, u64 seed, u64* dropped, unsigned* used /* [B][grid] */) {
  extern __shared__ __align__(32) unsigned char sm[];
  Rec* stage = reinterpret_cast<Rec*>(sm);                       // [B][NL][K]
  unsigned* tick = reinterpret_cast<unsigned*>(stage + (size_t)B * NL * K);
  unsigned* nline = tick + B;                                    // [B] lines flushed by this CTA
  unsigned* done = nline + B;                                    // [B][NL]
  volatile unsigned* lgen = done + NL * B;                       // [B][NL]
  for (int t = threadIdx.x; t < (2 + 2 * NL) * B; t += blockDim.x) tick[t] = 0;
  __syncthreads();
  const u64 tid = (u64)blockIdx.x * blockDim.x + threadIdx.x;
  u64 drop = 0;
  for (int it = 0; it < iters; ++it) {
    const u64 r = mix(seed + tid * 1315423911ull + (u64)it * 0x100000001B3ull);
    const int b = (int)(((r >> 32) * (u64)B) >> 32);
    const unsigned t = atomicAdd(&tick[b], 1u);
    const unsigned g = t / K, pos = t % K, line = g % NL, use = g / NL;
    Rec* ln = stage + ((size_t)b * NL + line) * K;
    bool pending = true;
    while (pending) {
      if (lgen[NL * b + line] == use) {
        ln[pos] = Rec{r | 1ull, r * 3ull, 1.0, 2.0};
        __threadfence_block();
        const unsigned d = atomicAdd(&done[NL * b + line], 1u);
        if (d == K - 1) {
          __threadfence_block();
          done[NL * b + line] = 0;
          const unsigned gl = atomicAdd(&nline[b], 1u);
          if (gl < cap_lines) {
            Rec* dst = pool + (((u64)b * gridDim.x + blockIdx.x) * cap_lines + gl) * K;
#pragma unroll
            for (int k = 0; k < K; ++k) { const Rec x = ln[k]; st256(dst + k, x.ka, x.kb, __double_as_longlong(x.v), __double_as_longlong(x.h)); }
          } else drop += K;
          __threadfence_block();
          lgen[NL * b + line] = use + 1;
        }
        pending = false;
      }
    }
  }
  __syncthreads();
  for (int b = threadIdx.x; b < B; b += blockDim.x) used[(size_t)b * gridDim.x + blockIdx.x] = nline[b];
  if (drop) atomicAdd(dropped, drop);
}
// A3: no staging: every CTA owns a private segment of each bin and appends with a shared-memory counter (no global atomic);
// consecutive records of a (bin, CTA) fill consecutive sectors, so L2 gets to combine them into full lines before write-back.
template <int U>
__global__ void __launch_bounds__(1024, 1)
append_private_kernel(Rec* pool, int B, unsigned cap_recs /* per (bin, CTA) */, int iters, u64 seed, u64* dropped, unsigned* used) {
  extern __shared__ __align__(32) unsigned char sm[];
  unsigned* cnt = reinterpret_cast<unsigned*>(sm);
  for (int t = threadIdx.x; t < B; t += blockDim.x) cnt[t] = 0;
  __syncthreads();
  const u64 tid = (u64)blockIdx.x * blockDim.x + threadIdx.x;
  u64 drop = 0;
  for (int it = 0; it < iters; it += U) {
    u64 r[U]; int b[U]; unsigned p[U];
#pragma unroll
    for (int u = 0; u < U; ++u) { r[u] = mix(seed + tid * 1315423911ull + (u64)(it + u) * 0x100000001B3ull); b[u] = (int)(((r[u] >> 32) * (u64)B) >> 32); }
#pragma unroll
    for (int u = 0; u < U; ++u) p[u] = atomicAdd(&cnt[b[u]], 1u);
#pragma unroll
    for (int u = 0; u < U; ++u) {
      if (p[u] < cap_recs) st256(pool + ((u64)b[u] * gridDim.x + blockIdx.x) * cap_recs + p[u], r[u] | 1ull, r[u] * 3ull, __double_as_longlong(1.0), __double_as_longlong(2.0));
      else ++drop;
    }
  }
  __syncthreads();
  for (int b = threadIdx.x; b < B; b += blockDim.x) used[(size_t)b * gridDim.x + blockIdx.x] = cnt[b];
  if (drop) atomicAdd(dropped, drop);
}
// A4: CTA-synchronous counting sort.  Warps append their records to a shared buffer (one shared atomic per warp, coalesced
// stores); when the buffer holds N records the CTA histograms them by bin, scans, scatters them into bin order in a second
// buffer and writes that out with consecutive threads on consecutive records, so every bin's run leaves as one or two
// line-sized requests into the CTA's private segment of the bin.
template <int N>
__global__ void __launch_bounds__(1024, 1)
part_sort_kernel(Rec* pool, int B, unsigned cap_recs /* per (bin, CTA) */, int rounds, u64 seed, u64* dropped, unsigned* used) {
  extern __shared__ __align__(32) unsigned char sm[];
  Rec* buf = reinterpret_cast<Rec*>(sm);                          // [N] arrival order
  Rec* srt = buf + N;                                            // [N] bin order
  unsigned* hist = reinterpret_cast<unsigned*>(srt + N);         // [B]
  unsigned* base = hist + B;                                     // [B] exclusive scan of hist
  unsigned* segu = base + B;                                     // [B] records this CTA has flushed per bin
  unsigned short* sbin = reinterpret_cast<unsigned short*>(segu + B);  // [N] bin of sorted position
  __shared__ unsigned fill, wtot[32];
  for (int t = threadIdx.x; t < B; t += blockDim.x) { hist[t] = 0; segu[t] = 0; }
  if (threadIdx.x == 0) fill = 0;
  __syncthreads();
  const u64 tid = (u64)blockIdx.x * blockDim.x + threadIdx.x;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  constexpr int PER = N / 1024;                                  // records per thread and round
  u64 drop = 0;
  for (int rd = 0; rd < rounds; ++rd) {
    // produce: every warp appends PER batches of 32 records
#pragma unroll
    for (int q = 0; q < PER; ++q) {
      const u64 r = mix(seed + tid * 1315423911ull + (u64)(rd * PER + q) * 0x100000001B3ull);
      unsigned pos = 0;
      if (lane == 0) pos = atomicAdd(&fill, 32u);
      pos = __shfl_sync(0xffffffffu, pos, 0) + lane;
      buf[pos] = Rec{r | 1ull, r * 3ull, 1.0, 2.0};
    }
    __syncthreads();
    // histogram + rank
    unsigned rk[PER]; int bn[PER];
#pragma unroll
    for (int q = 0; q < PER; ++q) {
      const u64 ka = buf[threadIdx.x + q * 1024].ka;
      bn[q] = (int)(((ka >> 32) * (u64)B) >> 32);
      rk[q] = atomicAdd(&hist[bn[q]], 1u);
    }
    __syncthreads();
    // exclusive scan of hist over B <= 1024 bins: one bin per thread
    {
      unsigned v = threadIdx.x < B ? hist[threadIdx.x] : 0u, x = v;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { unsigned y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
      if (lane == 31) wtot[warp] = x;
      __syncthreads();
      if (warp == 0) { unsigned w = wtot[lane], sx = w; for (int o = 1; o < 32; o <<= 1) { unsigned y = __shfl_up_sync(0xffffffffu, sx, o); if (lane >= o) sx += y; } wtot[lane] = sx - w; }
      __syncthreads();
      if (threadIdx.x < B) base[threadIdx.x] = wtot[warp] + x - v;
    }
    __syncthreads();
    // scatter into bin order
#pragma unroll
    for (int q = 0; q < PER; ++q) {
      const unsigned d = base[bn[q]] + rk[q];
      srt[d] = buf[threadIdx.x + q * 1024];
      sbin[d] = (unsigned short)bn[q];
    }
    __syncthreads();
    // write out: consecutive threads, consecutive records of a bin's run
#pragma unroll
    for (int q = 0; q < PER; ++q) {
      const int t = threadIdx.x + q * 1024;
      const int b = sbin[t];
      const unsigned p = segu[b] + ((unsigned)t - base[b]);
      const Rec x = srt[t];
      if (p < cap_recs) st256(pool + ((u64)b * gridDim.x + blockIdx.x) * cap_recs + p, x.ka, x.kb, __double_as_longlong(x.v), __double_as_longlong(x.h));
      else ++drop;
    }
    __syncthreads();
    if (threadIdx.x < B) { segu[threadIdx.x] += hist[threadIdx.x]; hist[threadIdx.x] = 0; }
    if (threadIdx.x == 0) fill = 0;
    __syncthreads();
  }
  for (int b = threadIdx.x; b < B; b += blockDim.x) used[(size_t)b * gridDim.x + blockIdx.x] = segu[b];
  if (drop) atomicAdd(dropped, drop);
}
// baseline: one global atomic + one scattered 32-byte store per record
__global__ void __launch_bounds__(1024, 1)
append_kernel(Rec* pool, u64* gcur, int B, u64 cap_recs, int iters, u64 seed, u64* dropped) {
  const u64 tid = (u64)blockIdx.x * blockDim.x + threadIdx.x;
  u64 drop = 0;
  for (int it = 0; it < iters; ++it) {
    const u64 r = mix(seed + tid * 1315423911ull + (u64)it * 0x100000001B3ull);
    const int b = (int)(((r >> 32) * (u64)B) >> 32);
    const u64 p = atomicAdd(&gcur[b], 1ull);
    if (p < cap_recs) st256(pool + (u64)b * cap_recs + p, r | 1ull, r * 3ull, __double_as_longlong(1.0), __double_as_longlong(2.0)); else ++drop;
  }
  if (drop) atomicAdd(dropped, drop);
}

// ------------------------------------------------------------------ B: one bin per CTA pass, deduplicated in shared memory
// bins: [nbins][M] records; keys inside a bin repeat `dup` times on average.  Table of record indices (short), 2M slots.
template <int M, int T>
__global__ void __launch_bounds__(T)
dedupe_kernel(const Rec* __restrict__ bins, int nbins, double e_s, double* out) {
  extern __shared__ __align__(32) unsigned char sm[];
  Rec* rec = reinterpret_cast<Rec*>(sm);                         // [M]
  int* tab = reinterpret_cast<int*>(rec + M);                    // [2M]
  __shared__ double wsum[32];
  double acc = 0.0;
  for (int bin = blockIdx.x; bin < nbins; bin += gridDim.x) {
    for (int t = threadIdx.x; t < 2 * M; t += blockDim.x) tab[t] = -1;
    const Rec* src = bins + (size_t)bin * M;
    for (int t = threadIdx.x; t < M; t += blockDim.x) { u64 a, b, c, d; ld256cs(src + t, a, b, c, d); rec[t] = Rec{a, b, __longlong_as_double(c), __longlong_as_double(d)}; }
    __syncthreads();
    for (int t = threadIdx.x; t < M; t += blockDim.x) {
      const u64 ka = rec[t].ka, kb = rec[t].kb;
      unsigned h = (unsigned)(mix(ka ^ (kb * 0x9E3779B97F4A7C15ull)) >> 40) & (2 * M - 1);
      for (;;) {
        const int cur = atomicCAS(&tab[h], -1, t);
        if (cur == -1) break;                                   // t represents its key
        if (rec[cur].ka == ka && rec[cur].kb == kb) { atomicAdd(&rec[cur].v, rec[t].v); rec[t].h = __longlong_as_double(0x7ff8000000000001ll); break; }
        h = (h + 1) & (2 * M - 1);
      }
    }
    __syncthreads();
    for (int t = threadIdx.x; t < M; t += blockDim.x) {
      const double hh = rec[t].h;
      if (hh == hh) { const double v = rec[t].v; acc += v * v / (e_s - hh); }
    }
    __syncthreads();
  }
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) { double s = 0; for (int w = 0; w < T / 32; ++w) s += wsum[w]; atomicAdd(out, s); }
}
__global__ void fill_bins_kernel(Rec* bins, u64 n, int M, int dup, u64 seed) {
  for (u64 t = (u64)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (u64)gridDim.x * blockDim.x) {
    const u64 bin = t / M;
    const u64 id = mix(seed + t) % (u64)(M / dup);              // M/dup distinct keys per bin
    const u64 k = mix(bin * 0x51ull + id * 0x1234567ull);
    bins[t] = Rec{k | 1ull, mix(k), 1.0 + (double)(t & 7), -2.0 - (double)(id & 15)};
  }
}

// ------------------------------------------------------------------ C: region-ordered merge into a big table
// Record r belongs to region r / per_region; its slot is inside that region of the table.  CTAs take chunks of records in
// order, so at any time the probes of the whole GPU fall into a window of a few regions (L2-resident), with no barrier.
__global__ void fill_ordered_kernel(Rec* recs, u64 n, u64 per_region, int dup, u64 seed) {
  for (u64 t = (u64)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (u64)gridDim.x * blockDim.x) {
    const u64 reg = t / per_region;
    const u64 id = mix(seed + t) % (per_region / dup);
    const u64 k = mix(reg * 0x9E37ull + id * 0x1234567ull);
    recs[t] = Rec{k | 1ull, mix(k), 1.0, -3.0};
  }
}
__global__ void __launch_bounds__(1024, 2)
merge_kernel(const Rec* __restrict__ recs, u64 n, u64 per_region, Rec* table, u64 region_slots, u64* cursor, int* overflow) {
  __shared__ u64 base;
  constexpr u64 kChunk = 8192;
  for (;;) {
    __syncthreads();
    if (threadIdx.x == 0) base = atomicAdd(cursor, kChunk);
    __syncthreads();
    const u64 b0 = base;
    if (b0 >= n) break;
    for (u64 t = b0 + threadIdx.x; t < b0 + kChunk && t < n; t += blockDim.x) {
      u64 ka, kb, vv, hh;
      ld256cs(recs + t, ka, kb, vv, hh);
      const u64 reg = t / per_region;
      u64 s = __umul64hi(mix(ka ^ kb), region_slots);
      Rec* tb = table + reg * region_slots;
      for (int probes = 0;; ++probes) {
        u64 a, b, c, d;
        ld256(tb + s, a, b, c, d);
        if (a == ka && b == kb) { atomicAdd(&tb[s].v, __longlong_as_double(vv)); break; }
        if ((a | b) == 0ull) {
          cas128(tb + s, ka, kb, a, b);
          if ((a | b) == 0ull) { tb[s].h = __longlong_as_double(hh); atomicAdd(&tb[s].v, __longlong_as_double(vv)); break; }
          if (a == ka && b == kb) { atomicAdd(&tb[s].v, __longlong_as_double(vv)); break; }
        }
        if (++s == region_slots) s = 0;
        if (probes > 100000) { *overflow = 1; break; }
      }
    }
  }
}

template <class F> float timed(F f) {
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  cudaEventRecord(e0); f(); cudaEventRecord(e1); cudaEventSynchronize(e1);
  float ms = 0; cudaEventElapsedTime(&ms, e0, e1); CK(cudaGetLastError());
  return ms;
}

template <int K> void run_part(int B, Rec* pool, u64 pool_recs, u64* gcur, u64* dropped, int sms) {
  const int iters = 2048;
  const u64 total = (u64)sms * 1024 * iters;
  const u64 cap_lines = pool_recs / B / K;
  const size_t smem = (size_t)B * 2 * K * sizeof(Rec) + 5 * (size_t)B * sizeof(unsigned);
  CK(cudaFuncSetAttribute(part_kernel<K>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  for (int rep = 0; rep < 2; ++rep) {
    CK(cudaMemset(gcur, 0, B * sizeof(u64))); CK(cudaMemset(dropped, 0, 8));
    float ms = timed([&] { part_kernel<K><<<sms, 1024, smem>>>(pool, gcur, B, cap_lines, iters, 77 + rep, dropped); });
    u64 d = 0; CK(cudaMemcpy(&d, dropped, 8, cudaMemcpyDeviceToHost));
    if (rep) printf("A staged  B=%5d K=%d (line %3d B, smem %3zu KB): %7.2f G rec/s  %6.2f TB/s  dropped %llu\n", B, K, K * 32, smem >> 10, total / (ms * 1e6), total * 32 / (ms * 1e9), d);
  }
}
template <int K, int NL> void run_part_private(int B, Rec* pool, u64 pool_recs, unsigned* used, u64* dropped, int sms) {
  const int iters = 2048;
  const u64 total = (u64)sms * 1024 * iters;
  const u64 cap_lines = pool_recs / B / sms / K;
  const size_t smem = (size_t)B * NL * K * sizeof(Rec) + (2 + 2 * NL) * (size_t)B * sizeof(unsigned);
  CK(cudaFuncSetAttribute(part_private_kernel<K, NL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  for (int rep = 0; rep < 2; ++rep) {
    CK(cudaMemset(dropped, 0, 8));
    float ms = timed([&] { part_private_kernel<K, NL><<<sms, 1024, smem>>>(pool, B, cap_lines, iters, 77 + rep, dropped, used); });
    u64 d = 0; CK(cudaMemcpy(&d, dropped, 8, cudaMemcpyDeviceToHost));
    if (rep) printf("A2 private B=%5d K=%d NL=%d (line %3d B, smem %3zu KB): %7.2f G rec/s  %6.2f TB/s  dropped %llu\n", B, K, NL, K * 32, smem >> 10, total / (ms * 1e6), total * 32 / (ms * 1e9), d);
  }
}
template <int U> void run_append_private(int B, Rec* pool, u64 pool_recs, unsigned* used, u64* dropped, int sms) {
  const int iters = 2048;
  const u64 total = (u64)sms * 1024 * iters;
  const unsigned cap = (unsigned)(pool_recs / B / sms);
  const size_t smem = (size_t)B * sizeof(unsigned);
  CK(cudaFuncSetAttribute(append_private_kernel<U>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  for (int rep = 0; rep < 2; ++rep) {
    CK(cudaMemset(dropped, 0, 8));
    float ms = timed([&] { append_private_kernel<U><<<sms, 1024, smem>>>(pool, B, cap, iters, 77 + rep, dropped, used); });
    u64 d = 0; CK(cudaMemcpy(&d, dropped, 8, cudaMemcpyDeviceToHost));
    if (rep) printf("A3 private append B=%5d U=%d (open lines %.1f MB): %7.2f G rec/s  %6.2f TB/s  dropped %llu\n", B, U, (double)B * sms * 128 / 1048576.0, total / (ms * 1e6), total * 32 / (ms * 1e9), d);
  }
}
template <int N> void run_part_sort(int B, Rec* pool, u64 pool_recs, unsigned* used, u64* dropped, int sms) {
  const int rounds = 2048 * 1024 / N;
  const u64 total = (u64)sms * N * rounds;
  const unsigned cap = (unsigned)(pool_recs / B / sms);
  const size_t smem = 2 * (size_t)N * sizeof(Rec) + 3 * (size_t)B * sizeof(unsigned) + (size_t)N * sizeof(unsigned short);
  CK(cudaFuncSetAttribute(part_sort_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  for (int rep = 0; rep < 2; ++rep) {
    CK(cudaMemset(dropped, 0, 8));
    float ms = timed([&] { part_sort_kernel<N><<<sms, 1024, smem>>>(pool, B, cap, rounds, 77 + rep, dropped, used); });
    u64 d = 0; CK(cudaMemcpy(&d, dropped, 8, cudaMemcpyDeviceToHost));
    if (rep) printf("A4 counting sort B=%5d N=%d (avg run %5.1f rec, smem %3zu KB): %7.2f G rec/s  %6.2f TB/s  dropped %llu\n", B, N, (double)N / B, smem >> 10, total / (ms * 1e6), total * 32 / (ms * 1e9), d);
  }
}
void run_append(int B, Rec* pool, u64 pool_recs, u64* gcur, u64* dropped, int sms) {
  const int iters = 2048;
  const u64 total = (u64)sms * 1024 * iters;
  for (int rep = 0; rep < 2; ++rep) {
    CK(cudaMemset(gcur, 0, B * sizeof(u64))); CK(cudaMemset(dropped, 0, 8));
    float ms = timed([&] { append_kernel<<<sms * 2, 1024>>>(pool, gcur, B, pool_recs / B, iters / 2, 77 + rep, dropped); });
    if (rep) printf("A append  B=%5d                          : %7.2f G rec/s  %6.2f TB/s\n", B, total / (ms * 1e6), total * 32 / (ms * 1e9));
  }
}
template <int M, int T> void run_dedupe(Rec* buf, u64 buf_recs, int dup, double* out, int sms) {
  const int nbins = (int)(buf_recs / M);
  fill_bins_kernel<<<sms * 8, 256>>>(buf, (u64)nbins * M, M, dup, 5); CK(cudaDeviceSynchronize());
  const size_t smem = (size_t)M * sizeof(Rec) + 2 * (size_t)M * sizeof(int);
  CK(cudaFuncSetAttribute(dedupe_kernel<M, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int per_sm = 0; CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, dedupe_kernel<M, T>, T, smem));
  for (int rep = 0; rep < 2; ++rep) {
    CK(cudaMemset(out, 0, 8));
    float ms = timed([&] { dedupe_kernel<M, T><<<sms * per_sm, T, smem>>>(buf, nbins, 1.0, out); });
    double s = 0; CK(cudaMemcpy(&s, out, 8, cudaMemcpyDeviceToHost));
    if (rep) printf("B dedupe  M=%5d T=%4d x %d CTAs/SM dup=%d (smem %3zu KB, %d bins): %7.2f G rec/s  %6.2f TB/s  sum %.6e\n", M, T, per_sm, dup, smem >> 10, nbins, (double)nbins * M / (ms * 1e6), (double)nbins * M * 32 / (ms * 1e9), s);
  }
}
void run_merge(Rec* recs, u64 n, Rec* table, u64 table_slots, u64 region_bytes, int dup, u64* cursor, int* overflow, int sms) {
  const u64 region_slots = region_bytes / 32;
  const u64 nreg = table_slots / region_slots;
  const u64 per_region = n / nreg;                               // load = per_region / dup / region_slots
  fill_ordered_kernel<<<sms * 8, 256>>>(recs, per_region * nreg, per_region, dup, 9); CK(cudaDeviceSynchronize());
  CK(cudaMemset(table, 0, table_slots * 32)); CK(cudaMemset(cursor, 0, 8)); CK(cudaMemset(overflow, 0, 4));
  float ms = timed([&] { merge_kernel<<<sms * 2, 1024>>>(recs, per_region * nreg, per_region, table, region_slots, cursor, overflow); });
  int ov = 0; CK(cudaMemcpy(&ov, overflow, 4, cudaMemcpyDeviceToHost));
  printf("C merge   region %7.1f MB (%llu regions, load %.2f, dup %d): %7.2f G rec/s%s\n", region_bytes / 1048576.0, nreg,
         (double)per_region / dup / region_slots, dup, (double)per_region * nreg / (ms * 1e6), ov ? "  OVERFLOW" : "");
}

int main(int argc, char** argv) {
  const char* sel = argc > 1 ? argv[1] : "abcsdef";  // a staged, b private staged, c private append, s counting sort, d append, e dedupe, f merge
  auto on = [&](char c) { for (const char* q = sel; *q; ++q) if (*q == c) return true; return false; };
  cudaDeviceProp prop; CK(cudaGetDeviceProperties(&prop, 0));
  const int sms = prop.multiProcessorCount;
  printf("%s, %d SMs, L2 %d MB\n", prop.name, sms, prop.l2CacheSize >> 20);
  const u64 pool_recs = 1ull << 29;                              // 16 GB of records
  Rec* pool; CK(cudaMalloc(&pool, pool_recs * 32));
  u64 *gcur, *dropped, *cursor; int* overflow; double* out;
  CK(cudaMalloc(&gcur, 65536 * 8)); CK(cudaMalloc(&dropped, 8)); CK(cudaMalloc(&cursor, 8)); CK(cudaMalloc(&overflow, 4)); CK(cudaMalloc(&out, 8));
  if (on('a')) {
    for (int B : {256, 512, 768}) run_part<4>(B, pool, pool_recs, gcur, dropped, sms);
    for (int B : {512, 1024, 1536}) run_part<2>(B, pool, pool_recs, gcur, dropped, sms);
  }
  unsigned* used; CK(cudaMalloc(&used, 16384 * 256 * 4));
  if (on('b')) {
  for (int B : {256, 512, 768}) run_part_private<4, 2>(B, pool, pool_recs, used, dropped, sms);
  for (int B : {128, 256, 384}) run_part_private<4, 4>(B, pool, pool_recs, used, dropped, sms);
  for (int B : {512, 1024, 1408}) run_part_private<2, 2>(B, pool, pool_recs, used, dropped, sms);
  for (int B : {256, 512, 704}) run_part_private<2, 4>(B, pool, pool_recs, used, dropped, sms);
  }
  if (on('c')) {
  for (int B : {256, 1024, 2048, 4096, 16384}) run_append_private<1>(B, pool, pool_recs, used, dropped, sms);
  for (int B : {256, 1024, 2048, 4096, 16384}) run_append_private<4>(B, pool, pool_recs, used, dropped, sms);
  }
  if (on('s')) {
    for (int B : {128, 256, 512, 1024}) run_part_sort<2048>(B, pool, pool_recs, used, dropped, sms);
    for (int B : {128, 256, 512, 1024}) run_part_sort<3072>(B, pool, pool_recs, used, dropped, sms);
    for (int B : {128, 256, 512}) run_part_sort<1024>(B, pool, pool_recs, used, dropped, sms);
  }
  if (on('d')) for (int B : {512, 2048, 16384}) run_append(B, pool, pool_recs, gcur, dropped, sms);
  if (on('e')) for (int dup : {1, 2, 4}) {
    run_dedupe<1024, 1024>(pool, 1ull << 27, dup, out, sms); run_dedupe<2048, 1024>(pool, 1ull << 27, dup, out, sms); run_dedupe<4096, 1024>(pool, 1ull << 27, dup, out, sms);
    run_dedupe<1024, 512>(pool, 1ull << 27, dup, out, sms); run_dedupe<2048, 512>(pool, 1ull << 27, dup, out, sms); run_dedupe<1024, 256>(pool, 1ull << 27, dup, out, sms);
  }
  if (!on('f')) return 0;
  const u64 table_slots = 1ull << 30;                            // 32 GB table
  Rec* table; CK(cudaMalloc(&table, table_slots * 32));
  for (int dup : {2, 4})
    for (u64 mb : {4ull, 16ull, 32ull, 64ull, 256ull, 32768ull}) run_merge(pool, pool_recs, table, table_slots, mb << 20, dup, cursor, overflow, sms);
  return 0;
}
