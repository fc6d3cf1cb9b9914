// probe: DRAM bytes fetched per random 32-byte read, by load flavour
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
typedef unsigned long long u64;
struct __align__(32) Slot { u64 ka, kb; double v, h; };
__device__ __forceinline__ u64 mix(u64 x) { x += 0x9E3779B97F4A7C15ull; x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull; x = (x ^ (x >> 27)) * 0x94D049BB133111EBull; return x ^ (x >> 31); }
template <int V> __device__ __forceinline__ u64 load32(const Slot* p, u64* sm) {
  u64 a, b, c, d;
  if (V == 0) { asm volatile("ld.relaxed.gpu.global.v4.u64 {%0,%1,%2,%3}, [%4];" : "=l"(a), "=l"(b), "=l"(c), "=l"(d) : "l"(p) : "memory"); return a + b + c + d; }
  if (V == 1) { asm volatile("ld.relaxed.gpu.global.L2::64B.v4.u64 {%0,%1,%2,%3}, [%4];" : "=l"(a), "=l"(b), "=l"(c), "=l"(d) : "l"(p) : "memory"); return a + b + c + d; }
  if (V == 2) { asm volatile("ld.global.nc.L1::no_allocate.v2.u64 {%0,%1}, [%2];" : "=l"(a), "=l"(b) : "l"(p)); asm volatile("ld.global.nc.L1::no_allocate.v2.u64 {%0,%1}, [%2+16];" : "=l"(c), "=l"(d) : "l"(p)); return a + b + c + d; }
  if (V == 3) {  // cp.async 16 B x 2 into shared memory
    unsigned s = (unsigned)__cvta_generic_to_shared(sm);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(p) : "memory");
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s + 16), "l"((const char*)p + 16) : "memory");
    asm volatile("cp.async.commit_group;" ::: "memory");
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    return sm[0] + sm[1] + sm[2] + sm[3];
  }
  if (V == 4) { asm volatile("ld.global.cs.v4.u64 {%0,%1,%2,%3}, [%4];" : "=l"(a), "=l"(b), "=l"(c), "=l"(d) : "l"(p) : "memory"); return a + b + c + d; }
  if (V == 5) { asm volatile("ld.global.L1::no_allocate.L2::evict_first.v4.u64 {%0,%1,%2,%3}, [%4];" : "=l"(a), "=l"(b), "=l"(c), "=l"(d) : "l"(p) : "memory"); return a + b + c + d; }
  if (V == 6) { asm volatile("ld.volatile.global.v4.u64 {%0,%1,%2,%3}, [%4];" : "=l"(a), "=l"(b), "=l"(c), "=l"(d) : "l"(p) : "memory"); return a + b + c + d; }
  return 0;
}
template <int V>
__global__ void k(const Slot* t, u64 cap, int iters, u64 seed, u64* sink) {
  __shared__ __align__(32) u64 sm[256 * 4];
  u64 tid = (u64)blockIdx.x * blockDim.x + threadIdx.x, acc = 0;
  for (int it = 0; it < iters; ++it) {
    u64 r = mix(seed + tid * 1315423911ull + (u64)it * 0x100000001B3ull);
    acc += load32<V>(t + __umul64hi(r, cap), sm + 4 * threadIdx.x);
  }
  if (acc == 0x1234567ull) *sink = acc;
}
int main() {
  const u64 cap = 1ull << 28;
  Slot* t; cudaMalloc(&t, cap * 32); cudaMemset(t, 0, cap * 32);
  u64* sink; cudaMalloc(&sink, 8);
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int grid = 148 * 8, block = 256, iters = (int)((1ull << 28) / ((u64)grid * block));
  float ms;
#define RUN(V) cudaEventRecord(e0); k<V><<<grid, block>>>(t, cap, iters, 7 + V, sink); cudaEventRecord(e1); cudaEventSynchronize(e1); cudaEventElapsedTime(&ms, e0, e1); \
  printf("variant %d : %7.2f Gops/s  (%s)\n", V, (double)iters * grid * block / (ms * 1e-3) / 1e9, cudaGetErrorString(cudaGetLastError()));
  RUN(0) RUN(1) RUN(2) RUN(3) RUN(4) RUN(5) RUN(6)
  return 0;
}
