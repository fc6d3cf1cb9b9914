// pt2 (a8, a9): external-determinant deduplication in an HBM open-addressing hash on 128-bit keys and the
// Epstein-Nesbet reduction (Eq. 13 second term; screening Eq. 14 / PAPER.md:219-227).
#include <math.h>

#include "enumerate.cuh"

EnumParams dh_make_params(detham_ctx* c, const HbLists* L);

namespace {

constexpr int kWarpsPerCta = 8;
constexpr int kFine = 1 << DH_MAX_PBITS;  // finest class histogram
constexpr int kProbeLimit = 1 << 16;

// one 32-byte sector per external: key, v_a = sum_i H_ai psi_i, H_aa.  Members of S are pre-inserted with v = NaN.
struct __align__(32) Slot { u64 ka, kb; double v, haa; };

__device__ __forceinline__ double member_flag() { return __longlong_as_double(0x7ff8000000000001ll); }

// ---------------------------------------------------------------- class histogram (pass planning)
struct CountSink {
  static constexpr bool kLookupFirst = true;  // singles are counted (upper bound) without being evaluated
  unsigned* hist;
  __device__ __forceinline__ bool pre(u64, u64, u64 z) { atomicAdd(hist + ((unsigned)z & (kFine - 1)), 1u); return false; }
  __device__ __forceinline__ void emit(bool act, u64, u64, u64 z, double, int, int, int, int, int, int) {
    if (act) atomicAdd(hist + ((unsigned)z & (kFine - 1)), 1u);
  }
};

__global__ void __launch_bounds__(kWarpsPerCta * 32)
count_kernel(EnumParams P, const u64* __restrict__ dets, const double* __restrict__ psi, int64_t nd, double eps2,
             u64* counters, u64* __restrict__ hist) {
  extern __shared__ __align__(16) unsigned char smem[];
  CtaTables T = dh_cta_stage(P, smem);
  size_t off = (dh_cta_table_bytes(P.n) + 15) & ~(size_t)15;
  WarpScratch* wsp = reinterpret_cast<WarpScratch*>(smem + off);
  unsigned* sh = reinterpret_cast<unsigned*>(smem + off + kWarpsPerCta * sizeof(WarpScratch));
  for (int t = threadIdx.x; t < kFine; t += blockDim.x) sh[t] = 0;
  __syncthreads();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  WarpScratch& ws = wsp[warp];
  CountSink sink{sh};
  for (;;) {
    u64 row = 0;
    if (lane == 0) row = atomicAdd(counters, 1ull);
    row = __shfl_sync(0xffffffffu, row, 0);
    if ((int64_t)row >= nd) break;
    const double p = psi[row];
    const u64 da = dets[2 * row], db = dets[2 * row + 1];
    u64 zsrc = 0;
    if (lane == 0) { zsrc = dh_zobrist(da, db, T.Z); atomicAdd(sh + ((unsigned)zsrc & (kFine - 1)), 1u); }
    zsrc = __shfl_sync(0xffffffffu, zsrc, 0);
    if (p == 0.0) continue;
    const double tau = eps2 == 0.0 ? 0.0 : __ddiv_rn(eps2, fabs(p));
    dh_fill_occ(P, ws, da, db, lane);
    dh_enumerate(P, T, ws, da, db, tau, zsrc, 0u, sink, lane);
    __syncwarp();
  }
  __syncthreads();
  for (int t = threadIdx.x; t < kFine; t += blockDim.x) if (sh[t]) atomicAdd(hist + t, (u64)sh[t]);
}

// ---------------------------------------------------------------- members of S of this pass's class
__global__ void member_insert_kernel(const u64* __restrict__ dets, int64_t nd, unsigned pmask, unsigned pass, Slot* table,
                                     u64 cap, int* overflow) {
  __shared__ u64 Z[128];
  for (int t = threadIdx.x; t < 128; t += blockDim.x) Z[t] = dh_zword(t);
  __syncthreads();
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nd) return;
  u64 a = dets[2 * t], b = dets[2 * t + 1];
  u64 z = dh_zobrist(a, b, Z);
  if (((unsigned)z & pmask) != pass) return;
  u64 slot = __umul64hi(z, cap);
  for (int probes = 0;; ++probes) {
    Slot* sp = table + slot;
    Key128 old = dh_cas128(sp, Key128{0ull, 0ull}, Key128{a, b});
    if (old.a == 0ull && old.b == 0ull) { sp->v = member_flag(); return; }
    if (++slot == cap) slot = 0;
    if (probes > kProbeLimit) { *overflow = 1; return; }
  }
}

// ---------------------------------------------------------------- accumulate
struct Pt2Sink {
  static constexpr bool kLookupFirst = false;
  Slot* table; u64 cap;
  const CtaTables* T; const WarpScratch* ws; int n;
  double psi, e0;
  u64 gen, contrib;
  int max_probe;
  int* overflow;
  __device__ __forceinline__ bool pre(u64, u64, u64) { return true; }
  __device__ __forceinline__ void emit(bool act, u64 ka, u64 kb, u64 z, double H, int kind, int s, int i, int j, int a, int b) {
    if (!act) return;
    ++gen;
    const double cval = H * psi;
    u64 slot = __umul64hi(z, cap);
    int probes = 0;
    for (;;) {
      Slot* sp = table + slot;
      u64 k0, k1, vb, hb;
      dh_ld256(sp, k0, k1, vb, hb);
      if (k0 == ka && k1 == kb) {
        if (vb != (u64)0x7ff8000000000001ull) { atomicAdd(&sp->v, cval); ++contrib; }  // not a member of S
        break;
      }
      if (k0 == 0ull && k1 == 0ull) {
        Key128 old = dh_cas128(sp, Key128{0ull, 0ull}, Key128{ka, kb});
        if (old.a == 0ull && old.b == 0ull) {  // claimed: this thread also records H_aa
          sp->haa = dh_excited_diag(*T, *ws, n, e0, kind, s, i, j, a, b);
          atomicAdd(&sp->v, cval);
          ++contrib;
          break;
        }
        if (old.a == ka && old.b == kb) { atomicAdd(&sp->v, cval); ++contrib; break; }  // lost the race to the same key
      }
      if (++slot == cap) slot = 0;
      if (++probes > kProbeLimit) { *overflow = 1; break; }
    }
    max_probe = max(max_probe, probes);
  }
};

__global__ void __launch_bounds__(kWarpsPerCta * 32)
pt2_accumulate_kernel(EnumParams P, const u64* __restrict__ dets, const double* __restrict__ psi, int64_t nd, double eps2,
                      unsigned pass, Slot* table, u64 cap, u64* counters /* [0] next row [1] gen [2] contrib [3] max probe */,
                      int* overflow) {
  extern __shared__ __align__(16) unsigned char smem[];
  CtaTables T = dh_cta_stage(P, smem);
  WarpScratch* wsp = reinterpret_cast<WarpScratch*>(smem + ((dh_cta_table_bytes(P.n) + 15) & ~(size_t)15));
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  WarpScratch& ws = wsp[warp];
  Pt2Sink sink{table, cap, &T, &ws, P.n, 0.0, 0.0, 0ull, 0ull, 0, overflow};
  for (;;) {
    u64 row = 0;
    if (lane == 0) row = atomicAdd(counters, 1ull);
    row = __shfl_sync(0xffffffffu, row, 0);
    if ((int64_t)row >= nd) break;
    const double p = psi[row];
    if (p == 0.0) continue;  // reading Q6: a source with zero amplitude generates nothing
    const double tau = eps2 == 0.0 ? 0.0 : __ddiv_rn(eps2, fabs(p));
    const u64 da = dets[2 * row], db = dets[2 * row + 1];
    dh_fill_occ(P, ws, da, db, lane);
    sink.psi = p;
    sink.e0 = dh_fill_U(P, T, ws, lane);
    u64 zsrc = 0;
    if (lane == 0) zsrc = dh_zobrist(da, db, T.Z);
    zsrc = __shfl_sync(0xffffffffu, zsrc, 0);
    dh_enumerate(P, T, ws, da, db, tau, zsrc, pass, sink, lane);
    __syncwarp();
  }
  u64 g = sink.gen, ct = sink.contrib;
  int mp = sink.max_probe;
  for (int o = 16; o > 0; o >>= 1) {
    g += __shfl_xor_sync(0xffffffffu, g, o);
    ct += __shfl_xor_sync(0xffffffffu, ct, o);
    mp = max(mp, __shfl_xor_sync(0xffffffffu, mp, o));
  }
  if (lane == 0) {
    if (g) atomicAdd(counters + 1, g);
    if (ct) atomicAdd(counters + 2, ct);
    atomicMax(counters + 3, (u64)mp);
  }
}

// ---------------------------------------------------------------- reduce: sum_a v_a^2 / (E_S - H_aa), and clear the table
__global__ void __launch_bounds__(256)
pt2_scan_kernel(Slot* table, u64 cap, double e_s, double* __restrict__ part /* [grid][4]: sum, sum_abs, min_den, count */) {
  double sum = 0.0, sabs = 0.0, mden = INFINITY, cnt = 0.0;
  for (u64 t = (u64)blockIdx.x * blockDim.x + threadIdx.x; t < cap; t += (u64)gridDim.x * blockDim.x) {
    struct { u64 x, y, z, w; } q;
    dh_ld256_cs(table + t, q.x, q.y, q.z, q.w);
    if (q.x | q.y) {
      if (q.z != (u64)0x7ff8000000000001ull) {
        double v = __longlong_as_double((long long)q.z), den = e_s - __longlong_as_double((long long)q.w);
        double term = v * v / den;
        sum += term; sabs += fabs(term); mden = fmin(mden, fabs(den)); cnt += 1.0;
      }
      dh_st256_zero(table + t);
    }
  }
  __shared__ double sh[4][8];
  for (int o = 16; o > 0; o >>= 1) {
    sum += __shfl_xor_sync(0xffffffffu, sum, o); sabs += __shfl_xor_sync(0xffffffffu, sabs, o);
    mden = fmin(mden, __shfl_xor_sync(0xffffffffu, mden, o)); cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
  }
  if ((threadIdx.x & 31) == 0) { int w = threadIdx.x >> 5; sh[0][w] = sum; sh[1][w] = sabs; sh[2][w] = mden; sh[3][w] = cnt; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0, b = 0, m = INFINITY, n = 0;
    for (int w = 0; w < 8; ++w) { a += sh[0][w]; b += sh[1][w]; m = fmin(m, sh[2][w]); n += sh[3][w]; }
    double* o = part + 4 * (size_t)blockIdx.x;
    o[0] = a; o[1] = b; o[2] = m; o[3] = n;
  }
}

__global__ void final_reduce4_kernel(const double* __restrict__ part, int nblk, double* out) {
  __shared__ double s0[256], s1[256], s2[256], s3[256];
  double a = 0, b = 0, m = INFINITY, n = 0;
  for (int t = threadIdx.x; t < nblk; t += 256) { a += part[4 * t]; b += part[4 * t + 1]; m = fmin(m, part[4 * t + 2]); n += part[4 * t + 3]; }
  s0[threadIdx.x] = a; s1[threadIdx.x] = b; s2[threadIdx.x] = m; s3[threadIdx.x] = n;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if (threadIdx.x < s) {
      s0[threadIdx.x] += s0[threadIdx.x + s]; s1[threadIdx.x] += s1[threadIdx.x + s];
      s2[threadIdx.x] = fmin(s2[threadIdx.x], s2[threadIdx.x + s]); s3[threadIdx.x] += s3[threadIdx.x + s];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) { out[0] = s0[0]; out[1] = s1[0]; out[2] = s2[0]; out[3] = s3[0]; }
}

__global__ void norm2_kernel(const double* __restrict__ psi, int64_t nd, double* __restrict__ part) {
  double a = 0.0;
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < nd; t += (int64_t)gridDim.x * blockDim.x) a = fma(psi[t], psi[t], a);
  __shared__ double sh[8];
  for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = a;
  __syncthreads();
  if (threadIdx.x == 0) { double s = 0; for (int w = 0; w < 8; ++w) s += sh[w]; part[4 * blockIdx.x] = s; part[4 * blockIdx.x + 1] = 0; part[4 * blockIdx.x + 2] = INFINITY; part[4 * blockIdx.x + 3] = 0; }
}

// ---------------------------------------------------------------- test hooks
struct ConnSink {
  static constexpr bool kLookupFirst = false;
  u64* keys; double* h; int count; int lane;
  __device__ __forceinline__ bool pre(u64, u64, u64) { return true; }
  __device__ __forceinline__ void emit(bool act, u64 ka, u64 kb, u64, double H, int, int, int, int, int, int) {
    unsigned m = __ballot_sync(0xffffffffu, act);
    if (act) { int pos = count + __popc(m & ((1u << lane) - 1u)); keys[2 * pos] = ka; keys[2 * pos + 1] = kb; h[pos] = H; }
    count += __popc(m);
  }
};

__global__ void connections_kernel(EnumParams P, const u64* __restrict__ dets, int64_t row, double tau, u64* keys, double* h, int* n_out) {
  extern __shared__ __align__(16) unsigned char smem[];
  CtaTables T = dh_cta_stage(P, smem);
  WarpScratch& ws = *reinterpret_cast<WarpScratch*>(smem + ((dh_cta_table_bytes(P.n) + 15) & ~(size_t)15));
  const int lane = threadIdx.x;
  const u64 da = dets[2 * row], db = dets[2 * row + 1];
  dh_fill_occ(P, ws, da, db, lane);
  u64 zsrc = dh_zobrist(da, db, T.Z);
  ConnSink sink{keys, h, 0, lane};
  dh_enumerate(P, T, ws, da, db, tau, zsrc, 0u, sink, lane);
  if (lane == 0) *n_out = sink.count;
}

__global__ void diagonals_kernel(int n, const double* __restrict__ J, const double* __restrict__ JK, const double* __restrict__ hd,
                                 double e_core, const u64* __restrict__ dets, int64_t m, double* __restrict__ out) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= m) return;
  u64 a = dets[2 * t], b = dets[2 * t + 1];
  double one = 0.0, two = 0.0;
  for (int p = 0; p < n; ++p) {
    bool pa = (a >> p) & 1ull, pb = (b >> p) & 1ull;
    if (pa) one += hd[p];
    if (pb) one += hd[p];
    for (int q = 0; q < n; ++q) {
      bool qa = (a >> q) & 1ull, qb = (b >> q) & 1ull;
      if (pa && qa) two += JK[p * n + q];
      if (pb && qb) two += JK[p * n + q];
      if (pa && qb) two += J[p * n + q];
      if (pb && qa) two += J[p * n + q];
    }
  }
  out[t] = e_core + one + 0.5 * two;
}

}  // namespace

static dh_status ensure_table(detham_ctx* c, int64_t slots) {
  if (c->table && c->table_slots >= slots) return DH_OK;
  if (c->table) cudaFree(c->table);
  c->table = nullptr; c->table_slots = 0;
  DH_CUDA(c, cudaMalloc(&c->table, (size_t)slots * sizeof(Slot)));
  DH_CUDA(c, cudaMemsetAsync(c->table, 0, (size_t)slots * sizeof(Slot), c->stream));
  c->table_slots = slots;
  return DH_OK;
}

dh_status dh_pt2(detham_ctx* c, const double* psi, double e_s, double eps2, double* out) {
  const int64_t nd = c->nd;
  const size_t smem_base = ((dh_cta_table_bytes(c->n) + 15) & ~(size_t)15) + kWarpsPerCta * sizeof(WarpScratch);
  int64_t want = (nd + kWarpsPerCta - 1) / kWarpsPerCta;
  const int grid = (int)(want < (int64_t)c->sm_count * 4 ? want : (int64_t)c->sm_count * 4);
  dh_status st;
  u64* hp = reinterpret_cast<u64*>(c->pinned);

  // ---- plan: partition count and table capacity
  int pbits = 0;
  int64_t slots = c->cfg_table_slots;
  c->ctr.ms_pt2_plan = 0.0;
  if (c->cfg_parts > 0) { while ((1 << pbits) < c->cfg_parts) ++pbits; }
  if (c->cfg_parts == 0 || slots == 0) {
    const HbLists* L0 = nullptr;
    st = dh_get_lists(c, 0, &L0); if (st != DH_OK) return st;
    EnumParams P0 = dh_make_params(c, L0);
    size_t smem = smem_base + kFine * sizeof(unsigned);
    DH_CUDA(c, cudaFuncSetAttribute(count_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    DH_CUDA(c, cudaMemsetAsync(c->dcount, 0, 8 * sizeof(u64), c->stream));
    DH_CUDA(c, cudaMemsetAsync(c->hist, 0, kFine * sizeof(u64), c->stream));
    DH_TICK(c, 0);
    count_kernel<<<grid, kWarpsPerCta * 32, smem, c->stream>>>(P0, c->dets, psi, nd, eps2, c->dcount, reinterpret_cast<u64*>(c->hist));
    DH_CUDA(c, cudaGetLastError());
    DH_TICK(c, 1);
    std::vector<u64> hist(kFine);
    DH_CUDA(c, cudaMemcpyAsync(hist.data(), c->hist, kFine * sizeof(u64), cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(c, cudaStreamSynchronize(c->stream));
    c->ctr.ms_pt2_plan = dh_elapsed(c, 0, 1);
    size_t free_b = 0, total_b = 0;
    DH_CUDA(c, cudaMemGetInfo(&free_b, &total_b));
    int64_t max_slots = (int64_t)(((double)free_b + (double)c->table_slots * sizeof(Slot)) * 0.92 / sizeof(Slot));
    if (slots > 0) max_slots = slots;
    auto max_class = [&](int pb) {
      u64 m = 0;
      for (int cl = 0; cl < (1 << pb); ++cl) { u64 s = 0; for (int f = cl; f < kFine; f += (1 << pb)) s += hist[f]; if (s > m) m = s; }
      return (int64_t)m;
    };
    if (c->cfg_parts == 0) {
      pbits = 0;
      while (pbits < DH_MAX_PBITS && (double)max_class(pbits) > 0.7 * (double)max_slots) ++pbits;
      if ((double)max_class(pbits) > 0.7 * (double)max_slots) return DH_ETABLEFULL;
    }
    if (slots == 0) {
      int64_t need = (int64_t)((double)max_class(pbits) / 0.5) + 1024;
      slots = need < max_slots ? need : max_slots;
    }
  }
  st = ensure_table(c, slots); if (st != DH_OK) return st;
  Slot* table = reinterpret_cast<Slot*>(c->table);

  const HbLists* L = nullptr;
  st = dh_get_lists(c, pbits, &L); if (st != DH_OK) return st;
  EnumParams P = dh_make_params(c, L);
  DH_CUDA(c, cudaFuncSetAttribute(pt2_accumulate_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_base));

  const int nparts = 1 << pbits;
  const int sgrid = (int)(((slots + 255) / 256) < (int64_t)c->sm_count * 16 ? ((slots + 255) / 256) : (int64_t)c->sm_count * 16);
  st = dh_ensure_red(c, 4 * ((int64_t)sgrid + 64) + 4 * (int64_t)(nparts + 1)); if (st != DH_OK) return st;
  double* results = c->red;                        // [nparts + 1][4]; row nparts = psi^T psi
  double* part = c->red + 4 * (int64_t)(nparts + 1);
  int* overflow = reinterpret_cast<int*>(c->dcount + 8);
  DH_CUDA(c, cudaMemsetAsync(c->dcount, 0, 32 * sizeof(u64), c->stream));

  norm2_kernel<<<64, 256, 0, c->stream>>>(psi, nd, part);
  final_reduce4_kernel<<<1, 256, 0, c->stream>>>(part, 64, results + 4 * nparts);
  DH_CUDA(c, cudaGetLastError());

  u64 gen = 0, contrib = 0, max_probe = 0;
  double ms_accum = 0.0, ms_scan = 0.0;
  for (int pass = 0; pass < nparts; ++pass) {
    DH_CUDA(c, cudaMemsetAsync(c->dcount, 0, 4 * sizeof(u64), c->stream));
    DH_TICK(c, 2);
    member_insert_kernel<<<(unsigned)((nd + 255) / 256), 256, 0, c->stream>>>(c->dets, nd, (unsigned)(nparts - 1), (unsigned)pass, table, (u64)slots, overflow);
    pt2_accumulate_kernel<<<grid, kWarpsPerCta * 32, smem_base, c->stream>>>(P, c->dets, psi, nd, eps2, (unsigned)pass, table, (u64)slots, c->dcount, overflow);
    DH_TICK(c, 3);
    pt2_scan_kernel<<<sgrid, 256, 0, c->stream>>>(table, (u64)slots, e_s, part);
    final_reduce4_kernel<<<1, 256, 0, c->stream>>>(part, sgrid, results + 4 * pass);
    DH_CUDA(c, cudaGetLastError());
    DH_TICK(c, 4);
    DH_CUDA(c, cudaMemcpyAsync(hp, c->dcount, 4 * sizeof(u64), cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(c, cudaMemcpyAsync(hp + 4, overflow, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(c, cudaStreamSynchronize(c->stream));
    ms_accum += dh_elapsed(c, 2, 3); ms_scan += dh_elapsed(c, 3, 4);
    gen += hp[1]; contrib += hp[2]; if (hp[3] > max_probe) max_probe = hp[3];
    if (*reinterpret_cast<int*>(hp + 4)) return DH_ETABLEFULL;  // the scan above already cleared the table
  }
  std::vector<double> res(4 * (size_t)(nparts + 1));
  DH_CUDA(c, cudaMemcpyAsync(res.data(), results, res.size() * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  DH_CUDA(c, cudaStreamSynchronize(c->stream));
  const double norm2 = res[4 * (size_t)nparts];
  double sum = 0, sabs = 0, mden = INFINITY, cnt = 0;
  c->partials.assign(nparts, 0.0);
  for (int p = 0; p < nparts; ++p) {
    c->partials[p] = res[4 * p] / norm2;
    sum += res[4 * p]; sabs += res[4 * p + 1]; mden = fmin(mden, res[4 * p + 2]); cnt += res[4 * p + 3];
  }
  *out = sum / norm2;
  c->ctr.pt2_generated = (int64_t)gen;
  c->ctr.pt2_contrib = (int64_t)contrib;
  c->ctr.pt2_external = (int64_t)cnt;
  c->ctr.pt2_parts = nparts;
  c->ctr.pt2_max_probe = (int32_t)max_probe;
  c->ctr.pt2_table_slots = slots;
  c->ctr.pt2_sum_abs = sabs / norm2;
  c->ctr.pt2_min_abs_den = mden;
  c->ctr.ms_pt2_accum = ms_accum;
  c->ctr.ms_pt2_scan = ms_scan;
  return DH_OK;
}

dh_status dh_connections(detham_ctx* c, int64_t row, double tau, std::vector<u64>& keys, std::vector<double>& h) {
  const HbLists* L = nullptr;
  dh_status st = dh_get_lists(c, 0, &L); if (st != DH_OK) return st;
  EnumParams P = dh_make_params(c, L);
  const int64_t n = c->n, na = c->na, nb = c->nb;
  auto c2 = [](int64_t x) { return x * (x - 1) / 2; };
  int64_t cap = na * (n - na) + nb * (n - nb) + c2(na) * c2(n - na) + c2(nb) * c2(n - nb) + na * nb * (n - na) * (n - nb) + 32;
  u64* dk = nullptr; double* dh = nullptr; int* dn = nullptr;
  DH_CUDA(c, cudaMalloc(&dk, cap * 2 * sizeof(u64)));
  DH_CUDA(c, cudaMalloc(&dh, cap * sizeof(double)));
  DH_CUDA(c, cudaMalloc(&dn, sizeof(int)));
  size_t smem = ((dh_cta_table_bytes(c->n) + 15) & ~(size_t)15) + sizeof(WarpScratch);
  DH_CUDA(c, cudaFuncSetAttribute(connections_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  connections_kernel<<<1, 32, smem, c->stream>>>(P, c->dets, row, tau, dk, dh, dn);
  DH_CUDA(c, cudaGetLastError());
  int m = 0;
  DH_CUDA(c, cudaMemcpyAsync(&m, dn, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
  DH_CUDA(c, cudaStreamSynchronize(c->stream));
  keys.resize(2 * (size_t)m); h.resize(m);
  if (m) {
    DH_CUDA(c, cudaMemcpy(keys.data(), dk, 2 * (size_t)m * sizeof(u64), cudaMemcpyDeviceToHost));
    DH_CUDA(c, cudaMemcpy(h.data(), dh, (size_t)m * sizeof(double), cudaMemcpyDeviceToHost));
  }
  cudaFree(dk); cudaFree(dh); cudaFree(dn);
  return DH_OK;
}

dh_status dh_diagonals(detham_ctx* c, const u64* dets, int64_t m, double* out) {
  diagonals_kernel<<<(unsigned)((m + 127) / 128), 128, 0, c->stream>>>(c->n, c->J, c->JK, c->hd, c->e_core, dets, m, out);
  DH_CUDA(c, cudaGetLastError());
  return DH_OK;
}
