// probe: ceiling of random 32-byte-sector traffic on this GPU (loads, RED.F64, CAS.128) versus table size and MLP
#include <cstdio>
#include <cstdlib>
#include <cstdint>
#include <cuda_runtime.h>
typedef unsigned long long u64;
struct __align__(32) Slot { u64 ka, kb; double v, h; };
__device__ __forceinline__ u64 mix(u64 x) { x += 0x9E3779B97F4A7C15ull; x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull; x = (x ^ (x >> 27)) * 0x94D049BB133111EBull; return x ^ (x >> 31); }
__device__ __forceinline__ void ld256(const void* p, u64& a, u64& b, u64& c, u64& d) { asm volatile("ld.relaxed.gpu.global.v4.u64 {%0,%1,%2,%3}, [%4];" : "=l"(a), "=l"(b), "=l"(c), "=l"(d) : "l"(p) : "memory"); }
__device__ __forceinline__ void cas128(void* addr, u64 va, u64 vb, u64& oa, u64& ob) {
  asm volatile("{\n\t.reg .b128 c, v, o;\n\tmov.b128 c, {%2, %3};\n\tmov.b128 v, {%4, %5};\n\tatom.relaxed.gpu.global.cas.b128 o, [%6], c, v;\n\tmov.b128 {%0, %1}, o;\n\t}"
               : "=l"(oa), "=l"(ob) : "l"(0ull), "l"(0ull), "l"(va), "l"(vb), "l"(addr) : "memory");
}
template <int MODE, int U>
__global__ void k(Slot* t, u64 cap, int iters, u64 seed, u64* sink) {
  u64 tid = (u64)blockIdx.x * blockDim.x + threadIdx.x;
  u64 acc = 0;
  for (int it = 0; it < iters; ++it) {
    u64 s[U], a[U], b[U], c[U], d[U], e[U];
#pragma unroll
    for (int u = 0; u < U; ++u) { u64 r = mix(seed + tid * 1315423911ull + (u64)(it * U + u) * 0x100000001B3ull); s[u] = __umul64hi(r, cap); a[u] = r | 1; }
    if (MODE == 0 || MODE == 1 || MODE == 4 || MODE == 6) {
#pragma unroll
      for (int u = 0; u < U; ++u) {
        if (MODE == 6) { a[u] = *reinterpret_cast<volatile u64*>(&t[s[u]].ka); c[u] = 0; }
        else ld256(t + s[u], b[u], d[u], c[u], e[u]);
      }
#pragma unroll
      for (int u = 0; u < U; ++u) acc += c[u] + (MODE == 6 ? a[u] : b[u] + e[u]);
    }
    if (MODE == 1 || MODE == 2) {
#pragma unroll
      for (int u = 0; u < U; ++u) atomicAdd(&t[s[u]].v, 1.0);
    }
    if (MODE == 3 || MODE == 4) {
#pragma unroll
      for (int u = 0; u < U; ++u) cas128(t + s[u], a[u], 7ull, b[u], d[u]);
#pragma unroll
      for (int u = 0; u < U; ++u) { if ((b[u] | d[u]) == 0) t[s[u]].h = 1.0; atomicAdd(&t[s[u]].v, 1.0); }
    }
    if (MODE == 5) {
#pragma unroll
      for (int u = 0; u < U; ++u) acc += (u64)atomicAdd(&t[s[u]].v, 1.0);
    }
  }
  if (acc == 0x1234567ull) *sink = acc;
}
template <int MODE, int U>
double run(Slot* t, u64 cap, int grid, int block, u64 ops) {
  int iters = (int)(ops / ((u64)grid * block * U));
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  u64* sink; cudaMalloc(&sink, 8);
  k<MODE, U><<<grid, block>>>(t, cap, 2, 99, sink);
  cudaDeviceSynchronize();
  cudaEventRecord(e0);
  k<MODE, U><<<grid, block>>>(t, cap, iters, 12345, sink);
  cudaEventRecord(e1); cudaEventSynchronize(e1);
  float ms; cudaEventElapsedTime(&ms, e0, e1);
  cudaError_t err = cudaGetLastError(); if (err != cudaSuccess) printf("ERR %s\n", cudaGetErrorString(err));
  cudaFree(sink);
  return (double)iters * grid * block * U / (ms * 1e-3);
}
int main(int argc, char** argv) {
  int gran = argc > 1 ? atoi(argv[1]) : 0;
  if (gran) { cudaError_t e = cudaDeviceSetLimit(cudaLimitMaxL2FetchGranularity, (size_t)gran); printf("set L2 fetch gran %d -> %s\n", gran, cudaGetErrorString(e)); }
  size_t g = 0; cudaDeviceGetLimit(&g, cudaLimitMaxL2FetchGranularity); printf("L2 fetch granularity = %zu\n", g);
  const u64 caps[] = {1ull << 21, 1ull << 25, 1ull << 28, 1ull << 31, 5000000000ull};
  const char* names[] = {"ld256", "ld256+red", "red", "cas+st+red", "ld256+cas+st+red", "atom.ret", "ld64"};
  for (u64 cap : caps) {
    Slot* t; if (cudaMalloc(&t, cap * 32) != cudaSuccess) { printf("alloc fail %llu\n", cap); continue; }
    cudaMemset(t, 0, cap * 32);
    const u64 ops = 1ull << 29;
    printf("cap %llu slots (%.1f GB)\n", cap, cap * 32 / 1e9);
    for (int block : {256, 512}) {
      int grid = 148 * (1024 / block) * 2;  // 2048 threads per SM
      printf(" block %d grid %d\n", block, grid);
#define R(M, U) printf("  %-18s U=%d : %7.2f Gops/s\n", names[M], U, run<M, U>(t, cap, grid, block, ops) / 1e9);
      R(0, 1) R(0, 4) R(0, 8) R(6, 4) R(2, 1) R(2, 4) R(1, 4) R(5, 4)
      cudaMemset(t, 0, cap * 32);
      R(3, 4)
      cudaMemset(t, 0, cap * 32);
      R(4, 4)
      cudaMemset(t, 0, cap * 32);
    }
    cudaFree(t);
  }
  return 0;
}
