// Declarations shared by the two PT2 organisations (pt2.cu: hash table in HBM; pt2_stream.cu: records partitioned by
// key region and deduplicated in L2-resident tables).  Nothing here is used by oracle/.
#pragma once
#include <math.h>

#include "enumerate.cuh"

// one 32-byte sector per external: key, v_a = sum_i H_ai psi_i, H_aa.  The same layout serves as the contribution record
// {key, H_ai psi_i, H_aa} of the streamed organisation.
struct __align__(32) Slot { u64 ka, kb; double v, haa; };

constexpr int kProbeLimit = 1 << 16;

// H_DD from the determinant alone (no source, no update): E_core + sum_p h_pp + 1/2 sum_{p,q} [J or J-K], one thread
__device__ __forceinline__ double dh_diag_from_scratch(int n, const double* __restrict__ J, const double* __restrict__ JK,
                                                       const double* __restrict__ hd, double e_core, u64 a, u64 b) {
  double one = 0.0, two = 0.0;
  for (int p = 0; p < n; ++p) {
    bool pa = (a >> p) & 1ull, pb = (b >> p) & 1ull;
    if (pa) one += hd[p];
    if (pb) one += hd[p];
    if (!pa && !pb) continue;
    for (int q = 0; q < n; ++q) {
      bool qa = (a >> q) & 1ull, qb = (b >> q) & 1ull;
      if (pa && qa) two += JK[p * n + q];
      if (pb && qb) two += JK[p * n + q];
      if (pa && qb) two += J[p * n + q];
      if (pb && qa) two += J[p * n + q];
    }
  }
  return e_core + one + 0.5 * two;
}

// multiplicative mix of a key: positions a key inside a table region (the region itself comes from the partition word)
__device__ __forceinline__ unsigned dh_key_hash(u64 ka, u64 kb) {
  u64 h = ka * 0x9E3779B97F4A7C15ull + kb * 0xC2B2AE3D27D4EB4Full;
  h ^= h >> 29;
  h *= 0xBF58476D1CE4E5B9ull;
  return (unsigned)(h >> 32);
}
// Home slot of a key in the HBM table.  rshift == 0: mulhi(partition word, capacity).  Binned passes (rshift > 0, capacity a
// multiple of 2^rshift): region = mulhi(partition word, regions), position inside the region from the key itself, so that the
// merge - which knows a record's region - needs no partition word.
__device__ __forceinline__ u64 dh_table_slot(u64 z, u64 ka, u64 kb, u64 cap, int rshift) {
  if (rshift == 0) return __umul64hi(z, cap);
  return (__umul64hi(z, cap >> rshift) << rshift) | (u64)(dh_key_hash(ka, kb) >> (32 - rshift));
}

// reduce `nblk` rows of {sum, sum_abs, min_den, count} into out[4] (pt2.cu)
void dh_launch_final_reduce4(const double* part, int nblk, double* out, cudaStream_t stream);

// What the planner hands the streamed organisation (pt2_stream.cu) for one attempt at 2^pbits key partitions.
struct StreamPlan {
  int pbits;             // key partitions = 1 << pbits
  double est_records;    // upper estimate of the contributions of the fullest partition
  double est_distinct;   // estimate of its distinct externals (<= est_records); sizes the region tables
};

// Streamed PT2: returns DH_ETABLEFULL when a segment of the record pool or a region table overflowed (the caller retries
// with more partitions or runs the table organisation), DH_ENOMEM when the pool does not fit.
dh_status dh_pt2_stream(detham_ctx* c, const double* psi, double e_s, double eps2, const StreamPlan& plan, double* out);
