// probe: cost of "atomicAdd(cursor[bin]) + 32-byte store" appends versus bin count; TLB cliff of random loads vs footprint
#include <cstdio>
#include <cstdlib>
#include <cstdint>
#include <cuda_runtime.h>
typedef unsigned long long u64;
struct __align__(32) Rec { u64 a, b, c, d; };
__device__ __forceinline__ u64 mix(u64 x) { x += 0x9E3779B97F4A7C15ull; x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull; x = (x ^ (x >> 27)) * 0x94D049BB133111EBull; return x ^ (x >> 31); }
__device__ __forceinline__ void st256(void* p, u64 a, u64 b, u64 c, u64 d) { asm volatile("st.global.cs.v4.u64 [%0], {%1,%2,%3,%4};" ::"l"(p), "l"(a), "l"(b), "l"(c), "l"(d) : "memory"); }
__device__ __forceinline__ void ld256(const void* p, u64& a, u64& b, u64& c, u64& d) { asm volatile("ld.relaxed.gpu.global.v4.u64 {%0,%1,%2,%3}, [%4];" : "=l"(a), "=l"(b), "=l"(c), "=l"(d) : "l"(p) : "memory"); }
// MODE 0: atomic + store; 1: atomic only; 2: store only to pseudo-sequential position per bin (no atomic; position from iteration)
template <int MODE, int U>
__global__ void k(Rec* pool, unsigned* cursor, u64 nbins, u64 cap, int iters, u64 seed, u64* sink) {
  u64 tid = (u64)blockIdx.x * blockDim.x + threadIdx.x;
  u64 acc = 0;
  for (int it = 0; it < iters; ++it) {
    u64 bin[U]; unsigned off[U];
#pragma unroll
    for (int u = 0; u < U; ++u) { u64 r = mix(seed + tid * 1315423911ull + (u64)(it * U + u) * 0x100000001B3ull); bin[u] = __umul64hi(r, nbins); }
    if (MODE != 2) {
#pragma unroll
      for (int u = 0; u < U; ++u) off[u] = atomicAdd(cursor + bin[u], 1u);
    } else {
#pragma unroll
      for (int u = 0; u < U; ++u) off[u] = (unsigned)((tid * iters + it) * U + u) % (unsigned)cap;
    }
    if (MODE != 1) {
#pragma unroll
      for (int u = 0; u < U; ++u) if (off[u] < cap) st256(pool + bin[u] * cap + off[u], bin[u], off[u], tid, it);
    } else {
#pragma unroll
      for (int u = 0; u < U; ++u) acc += off[u];
    }
  }
  if (acc == 0x1234567ull) *sink = acc;
}
template <int U>
__global__ void rl(const Rec* t, u64 cap, int iters, u64 seed, u64* sink) {
  u64 tid = (u64)blockIdx.x * blockDim.x + threadIdx.x; u64 acc = 0;
  for (int it = 0; it < iters; ++it) {
    u64 a[U], b[U], c[U], d[U];
#pragma unroll
    for (int u = 0; u < U; ++u) { u64 r = mix(seed + tid * 1315423911ull + (u64)(it * U + u) * 0x100000001B3ull); ld256(t + __umul64hi(r, cap), a[u], b[u], c[u], d[u]); }
#pragma unroll
    for (int u = 0; u < U; ++u) acc += a[u] + b[u] + c[u] + d[u];
  }
  if (acc == 0x1234567ull) *sink = acc;
}
int main() {
  u64* sink; cudaMalloc(&sink, 8);
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  const u64 total = 3ull << 30;  // records of pool capacity (96 GB)
  Rec* pool; if (cudaMalloc(&pool, total * 32) != cudaSuccess) { printf("alloc fail\n"); return 1; }
  unsigned* cursor; cudaMalloc(&cursor, (1 << 22) * 4);
  const u64 ops = 1ull << 30;
  for (int block : {512}) {
    int grid = 148 * (2048 / block);
    for (u64 nbins : {256ull, 4096ull, 32768ull, 262144ull, 2097152ull}) {
      u64 cap = total / nbins;
      int iters = (int)(ops / ((u64)grid * block * 4));
      float ms;
#define RUN(M) cudaMemset(cursor, 0, nbins * 4); cudaEventRecord(e0); k<M, 4><<<grid, block>>>(pool, cursor, nbins, cap, iters, 777, sink); cudaEventRecord(e1); cudaEventSynchronize(e1); cudaEventElapsedTime(&ms, e0, e1); \
      printf("nbins %8llu mode %d : %7.2f Gops/s\n", nbins, M, (double)iters * grid * block * 4 / (ms * 1e-3) / 1e9);
      RUN(0) RUN(1) RUN(2)
    }
  }
  // TLB cliff: random 32-byte loads vs footprint
  for (double gb : {48.0, 64.0, 72.0, 80.0, 88.0, 96.0}) {
    u64 cap = (u64)(gb * 1e9 / 32);
    int grid = 148 * 4, block = 512; int iters = (int)((1ull << 29) / ((u64)grid * block * 4)); float ms;
    rl<4><<<grid, block>>>(pool, cap, 2, 1, sink); cudaDeviceSynchronize();
    cudaEventRecord(e0); rl<4><<<grid, block>>>(pool, cap, iters, 5, sink); cudaEventRecord(e1); cudaEventSynchronize(e1); cudaEventElapsedTime(&ms, e0, e1);
    printf("random ld256 footprint %5.0f GB : %7.2f Gops/s\n", gb, (double)iters * grid * block * 4 / (ms * 1e-3) / 1e9);
  }
  cudaFree(pool);
  for (double gb : {104.0, 112.0, 120.0, 128.0, 144.0, 160.0}) {
    u64 cap = (u64)(gb * 1e9 / 32);
    Rec* t; if (cudaMalloc(&t, cap * 32) != cudaSuccess) { printf("alloc fail %f\n", gb); continue; }
    int grid = 148 * 4, block = 512; int iters = (int)((1ull << 29) / ((u64)grid * block * 4)); float ms;
    rl<4><<<grid, block>>>(t, cap, 2, 1, sink); cudaDeviceSynchronize();
    cudaEventRecord(e0); rl<4><<<grid, block>>>(t, cap, iters, 5, sink); cudaEventRecord(e1); cudaEventSynchronize(e1); cudaEventElapsedTime(&ms, e0, e1);
    printf("random ld256 footprint %5.0f GB : %7.2f Gops/s\n", gb, (double)iters * grid * block * 4 / (ms * 1e-3) / 1e9);
    cudaFree(t);
  }
  return 0;
}
