// probe: scattered 32-byte record stores, instruction variants
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
typedef unsigned long long u64;
struct __align__(32) Rec { u64 a, b, c, d; };
__device__ __forceinline__ u64 mix(u64 x) { x += 0x9E3779B97F4A7C15ull; x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull; x = (x ^ (x >> 27)) * 0x94D049BB133111EBull; return x ^ (x >> 31); }
template <int V> __device__ __forceinline__ void store(Rec* p, u64 a, u64 b, u64 c, u64 d) {
  if (V == 0) asm volatile("st.global.cs.v4.u64 [%0], {%1,%2,%3,%4};" ::"l"(p), "l"(a), "l"(b), "l"(c), "l"(d) : "memory");
  if (V == 1) asm volatile("st.global.v4.u64 [%0], {%1,%2,%3,%4};" ::"l"(p), "l"(a), "l"(b), "l"(c), "l"(d) : "memory");
  if (V == 2) { asm volatile("st.global.cs.v2.u64 [%0], {%1,%2};" ::"l"(p), "l"(a), "l"(b) : "memory"); asm volatile("st.global.cs.v2.u64 [%0+16], {%1,%2};" ::"l"(p), "l"(c), "l"(d) : "memory"); }
  if (V == 3) { asm volatile("st.global.v2.u64 [%0], {%1,%2};" ::"l"(p), "l"(a), "l"(b) : "memory"); asm volatile("st.global.v2.u64 [%0+16], {%1,%2};" ::"l"(p), "l"(c), "l"(d) : "memory"); }
  if (V == 4) { p->a = a; p->b = b; p->c = c; p->d = d; }
  if (V == 5) { asm volatile("st.global.wt.v2.u64 [%0], {%1,%2};" ::"l"(p), "l"(a), "l"(b) : "memory"); asm volatile("st.global.wt.v2.u64 [%0+16], {%1,%2};" ::"l"(p), "l"(c), "l"(d) : "memory"); }
}
template <int V, int U>
__global__ void k(Rec* pool, unsigned* cursor, u64 nbins, u64 cap, int iters, u64 seed) {
  u64 tid = (u64)blockIdx.x * blockDim.x + threadIdx.x;
  for (int it = 0; it < iters; ++it) {
    u64 bin[U]; unsigned off[U];
#pragma unroll
    for (int u = 0; u < U; ++u) { u64 r = mix(seed + tid * 1315423911ull + (u64)(it * U + u) * 0x100000001B3ull); bin[u] = __umul64hi(r, nbins); }
#pragma unroll
    for (int u = 0; u < U; ++u) off[u] = atomicAdd(cursor + bin[u], 1u);
#pragma unroll
    for (int u = 0; u < U; ++u) if (off[u] < cap) store<V>(pool + bin[u] * cap + off[u], bin[u], off[u], tid, it);
  }
}
int main() {
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  for (double gb : {2.0, 32.0, 96.0}) {
    const u64 total = (u64)(gb * 1e9 / 32);
    Rec* pool; if (cudaMalloc(&pool, total * 32) != cudaSuccess) { printf("alloc fail\n"); return 1; }
    unsigned* cursor; cudaMalloc(&cursor, (1 << 22) * 4);
    for (u64 nbins : {4096ull, 32768ull}) {
      u64 cap = total / nbins;
      u64 ops = total * 3 / 4; if (ops > (1ull << 30)) ops = 1ull << 30;
      int grid = 148 * 4, block = 512; int iters = (int)(ops / ((u64)grid * block * 4)); float ms;
#define RUN(V) cudaMemset(cursor, 0, nbins * 4); cudaDeviceSynchronize(); cudaEventRecord(e0); k<V, 4><<<grid, block>>>(pool, cursor, nbins, cap, iters, 777); cudaEventRecord(e1); cudaEventSynchronize(e1); cudaEventElapsedTime(&ms, e0, e1); \
      printf("pool %4.0f GB nbins %6llu variant %d : %7.2f Gops/s\n", gb, nbins, V, (double)iters * grid * block * 4 / (ms * 1e-3) / 1e9);
      RUN(0) RUN(1) RUN(2) RUN(3) RUN(4) RUN(5)
    }
    cudaFree(pool); cudaFree(cursor);
  }
  return 0;
}
