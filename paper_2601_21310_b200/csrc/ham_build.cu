// Determinant store lookup (a1) and CSR H_SS construction (a6).  PAPER.md:206, 269.
#include "enumerate.cuh"

namespace {

constexpr int kWarpsPerCta = 8;    // row-sort kernels
constexpr int kBuildWarps = 16;    // build_kernel: 2 CTAs per SM share the staged tables; 64 registers -> 32 warps per SM

// ---------------------------------------------------------------- determinant store
__global__ void validate_kernel(const u64* __restrict__ dets, int64_t nd, int n, int na, int nb, int* flags) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nd) return;
  u64 a = dets[2 * t], b = dets[2 * t + 1];
  u64 hi = n == 64 ? 0ull : ~((1ull << n) - 1ull);
  if (__popcll(a) != na || __popcll(b) != nb || (a & hi) || (b & hi)) flags[1] = 1;
  if (t > 0) {
    u64 pa = dets[2 * t - 2], pb = dets[2 * t - 1];
    if (!(pa < a || (pa == a && pb < b))) flags[0] = 1;
  }
}

// L2-resident open-addressing index of S: slot = mulhi(z(D), cap), linear probing, EMPTY = {0,0}
__global__ void shash_insert_kernel(const u64* __restrict__ dets, int64_t nd, u64* keys, int* idx, u64 cap, unsigned* bits,
                                    u64 nbits) {
  __shared__ u64 Z[128];
  for (int t = threadIdx.x; t < 128; t += blockDim.x) Z[t] = dh_zword(t);
  __syncthreads();
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nd) return;
  u64 a = dets[2 * t], b = dets[2 * t + 1];
  const u64 z = dh_zobrist(a, b, Z);
  if (bits)  // membership pre-filter (dh_maybe_member): two bits of one 64-bit word per determinant; the index of P has none
    atomicOr(reinterpret_cast<u64*>(bits) + dh_filter_word(nbits, z), dh_filter_mask(z));
  u64 slot = __umul64hi(z, cap);
  for (;;) {
    Key128 old = dh_cas128(keys + 2 * slot, Key128{0ull, 0ull}, Key128{a, b});
    if (old.a == 0ull && old.b == 0ull) { idx[slot] = (int)t; return; }
    if (++slot == cap) slot = 0;
  }
}

// ---------------------------------------------------------------- CSR sinks
// Single-pass build: every warp appends the (column, value) hits of its rows to an arena in blocks of kBlk entries
// reserved with one atomic each; a row's hits form one or more segments {row, offset in row, arena offset, count}.
// After the pass the row counts are scanned and the segments copied to their CSR positions.  If the arena (sized from
// the previous build) is too small the pass keeps counting, and the host reruns it with the exact size.
constexpr int kBlk = 1024;
struct Seg { int row, local, cnt, pad; int64_t off; };

struct BuildSink {
  static constexpr bool kLookupFirst = true;
  static constexpr bool kLazySign = true;   // the phase of a double is worked out for the hits only
  u64 da, db;              // the row's determinant (for the lazy phase)
  const u64* keys; const int* idx; u64 cap;
  const unsigned* bits; u64 nbits;
  int* acol; double* aval; int64_t arena_cap;
  u64* cursors;            // [2] arena cursor, [3] segment cursor
  Seg* segs; int64_t seg_cap; int* overflow;
  int row;
  int count;               // warp-uniform running count of the row's hits
  int64_t wpos, wend;      // warp-uniform write window in the arena (wpos < 0: arena exhausted, count only)
  int64_t seg_start; int seg_local;
  u64 generated;           // per-lane count of screened candidates looked up
  int lane;
  int pre_tok;
  __device__ __forceinline__ void close_seg() {
    const int64_t m = wpos - seg_start;
    if (wpos >= 0 && m > 0 && lane == 0) {
      u64 s = atomicAdd(cursors + 3, 1ull);
      if ((int64_t)s < seg_cap) segs[s] = Seg{row, seg_local, (int)m, 0, seg_start};
      else *overflow = 1;
    }
  }
  __device__ __forceinline__ void begin_row(int r, u64 a, u64 b) { row = r; da = a; db = b; count = 0; seg_start = wpos; seg_local = 0; }
  __device__ __forceinline__ void end_row() { close_seg(); }
  __device__ __forceinline__ void put(bool has, int tok, double H) {
    const unsigned hit = __ballot_sync(0xffffffffu, has);
    if (!hit) return;
    const int h = __popc(hit);
    if (wpos >= 0 && wpos + h > wend) {  // block full: close the segment and reserve the next block
      close_seg();
      u64 b = 0;
      if (lane == 0) b = atomicAdd(cursors + 2, (u64)kBlk);
      b = __shfl_sync(0xffffffffu, b, 0);
      if ((int64_t)b + kBlk > arena_cap) { wpos = -1; if (lane == 0) *overflow = 1; }
      else { wpos = (int64_t)b; wend = wpos + kBlk; }
      seg_start = wpos; seg_local = count;
    }
    if (wpos >= 0) {
      if (has) { const int64_t pos = wpos + __popc(hit & ((1u << lane) - 1u)); DH_CHECK(pos >= 0 && pos < arena_cap); acol[pos] = tok; aval[pos] = H; }
      wpos += h;
    }
    count += h;
  }
  __device__ __forceinline__ bool pre(u64 ka, u64 kb, u64 z) {
    ++generated;
    pre_tok = (!bits || dh_maybe_member(bits, nbits, z)) ? dh_shash_find(keys, idx, cap, ka, kb, z) : -1;
    return pre_tok >= 0;
  }
  __device__ __forceinline__ void emit(bool act, u64 ka, u64 kb, u64 z, double H, int kind, int s, int i, int j, int a, int b) {
    int tok = -1;
    if (act) {
      if (kind == 0) tok = pre_tok;
      else {
        ++generated;
        if (!bits || dh_maybe_member(bits, nbits, z)) tok = dh_shash_find(keys, idx, cap, ka, kb, z);
        if (tok >= 0 && dh_double_parity(da, db, kind, s, i, j, a, b)) H = -H;
      }
    }
    put(tok >= 0, tok, H);
  }
};

// kSP = false: H_SS (a6): tau = eps for every row, diagonal first.  kSP = true: H_SP (row f3): the index is that of the caller's
// sorted P, tau_i = eps / |psi_i| as in pt2 / expand (reading Q6, Q9), rows with psi_i == 0 stay empty, no diagonal.
template <bool kSP>
__global__ void __launch_bounds__(kBuildWarps * 32, 2)
build_kernel(EnumParams P, const u64* __restrict__ dets, const double* __restrict__ psi, int64_t nd, double eps, const u64* __restrict__ hkeys,
             const int* __restrict__ hidx, u64 hcap, const unsigned* __restrict__ hbits, u64 hnbits, int* __restrict__ row_cnt, int* acol, double* aval, int64_t arena_cap,
             Seg* segs, int64_t seg_cap, u64* counters /* [0] next row [1] generated [2] arena cursor [3] segments */,
             int* overflow) {
  extern __shared__ __align__(16) unsigned char smem[];
  CtaTables T = dh_cta_stage(P, smem);
  WarpScratch* wsp = reinterpret_cast<WarpScratch*>(smem + ((dh_cta_table_bytes(P.n) + 15) & ~(size_t)15));
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  WarpScratch& ws = wsp[warp];
  BuildSink sink{0ull, 0ull, hkeys, hidx, hcap, hbits, hnbits, acol, aval, arena_cap, counters, segs, seg_cap, overflow, 0, 0, 0, 0, 0, 0, 0ull, lane, -1};
  for (;;) {
    u64 row = 0;
    if (lane == 0) row = atomicAdd(counters, 1ull);
    row = __shfl_sync(0xffffffffu, row, 0);
    if ((int64_t)row >= nd) break;
    const u64 da = dets[2 * row], db = dets[2 * row + 1];
    double tau = eps;
    if (kSP) {
      const double p = psi[row];
      if (p == 0.0) { if (lane == 0) row_cnt[row] = 0; continue; }
      tau = eps == 0.0 ? 0.0 : __ddiv_rn(eps, fabs(p));
    }
    dh_fill_occ(P, ws, da, db, lane);
    const double e0 = dh_fill_U(P, T, ws, lane);
    sink.begin_row((int)row, da, db);
    if (!kSP) sink.put(lane == 0, (int)row, e0);  // the diagonal is always kept (reading Q4)
    u64 zsrc = 0;
    if (lane == 0) zsrc = dh_zobrist(da, db, T.Z);
    zsrc = __shfl_sync(0xffffffffu, zsrc, 0);
    dh_enumerate(P, T, ws, da, db, tau, zsrc, 0u, sink, lane);
    sink.end_row();
    if (lane == 0) row_cnt[row] = sink.count;
    __syncwarp();
  }
  u64 gen = sink.generated;
  for (int o = 16; o > 0; o >>= 1) gen += __shfl_xor_sync(0xffffffffu, gen, o);
  if (lane == 0 && gen) atomicAdd(counters + 1, gen);
}

// Sink of the complete-the-sum pass (row f2, the alternative of reading Q9): every excitation of the source that is a key of
// P adds H_ai psi_i to v[position of a in P]; nothing is stored.
struct CompleteSink {
  static constexpr bool kLookupFirst = true;
  static constexpr bool kLazySign = true;   // the phase of a double is worked out for the keys of P only
  u64 da, db;
  const u64* keys; const int* idx; u64 cap;
  double* v;
  double psi_i;
  u64 generated;
  int pre_tok;
  __device__ __forceinline__ bool pre(u64 ka, u64 kb, u64 z) {
    ++generated;
    pre_tok = dh_shash_find(keys, idx, cap, ka, kb, z);
    return pre_tok >= 0;
  }
  __device__ __forceinline__ void emit(bool act, u64 ka, u64 kb, u64 z, double H, int kind, int s, int i, int j, int a, int b) {
    if (!act) return;
    int tok = pre_tok;
    if (kind != 0) {
      ++generated;
      tok = dh_shash_find(keys, idx, cap, ka, kb, z);
      if (tok >= 0 && dh_double_parity(da, db, kind, s, i, j, a, b)) H = -H;
    }
    if (tok >= 0) atomicAdd(v + tok, H * psi_i);
  }
};

// v[a] += sum_i H_ai psi_i over EVERY single and double excitation of every source with psi_i != 0 (tau = 0: the whole lists)
__global__ void __launch_bounds__(kBuildWarps * 32, 2)
complete_kernel(EnumParams P, const u64* __restrict__ dets, const double* __restrict__ psi, int64_t nd, const u64* __restrict__ hkeys,
                const int* __restrict__ hidx, u64 hcap, double* __restrict__ v, u64* counters /* [0] next row [1] looked up */) {
  extern __shared__ __align__(16) unsigned char smem[];
  CtaTables T = dh_cta_stage(P, smem);
  WarpScratch* wsp = reinterpret_cast<WarpScratch*>(smem + ((dh_cta_table_bytes(P.n) + 15) & ~(size_t)15));
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  WarpScratch& ws = wsp[warp];
  CompleteSink sink{0ull, 0ull, hkeys, hidx, hcap, v, 0.0, 0ull, -1};
  for (;;) {
    u64 row = 0;
    if (lane == 0) row = atomicAdd(counters, 1ull);
    row = __shfl_sync(0xffffffffu, row, 0);
    if ((int64_t)row >= nd) break;
    const double p = psi[row];
    if (p == 0.0) continue;
    const u64 da = dets[2 * row], db = dets[2 * row + 1];
    dh_fill_occ(P, ws, da, db, lane);
    const double e0 = dh_fill_U(P, T, ws, lane);
    sink.da = da; sink.db = db; sink.psi_i = p;
    u64 zsrc = 0;
    if (lane == 0) {
      zsrc = dh_zobrist(da, db, T.Z);
      const int self = dh_shash_find(hkeys, hidx, hcap, da, db, zsrc);  // a key list may hold members of S: the sum runs over i = a too
      if (self >= 0) atomicAdd(v + self, e0 * p);
    }
    zsrc = __shfl_sync(0xffffffffu, zsrc, 0);
    dh_enumerate(P, T, ws, da, db, 0.0, zsrc, 0u, sink, lane);
    __syncwarp();
  }
  u64 gen = sink.generated;
  for (int o = 16; o > 0; o >>= 1) gen += __shfl_xor_sync(0xffffffffu, gen, o);
  if (lane == 0 && gen) atomicAdd(counters + 1, gen);
}

// arena segments -> CSR positions, one warp per segment
__global__ void __launch_bounds__(256)
copy_segs_kernel(const Seg* __restrict__ segs, int64_t nseg, const int64_t* __restrict__ row_ptr, const int* __restrict__ acol,
                 const double* __restrict__ aval, int* __restrict__ col, double* __restrict__ val) {
  const int lane = threadIdx.x & 31;
  const int64_t nw = (int64_t)gridDim.x * (blockDim.x >> 5);
  for (int64_t s = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); s < nseg; s += nw) {
    const Seg g = segs[s];
    const int64_t dst = row_ptr[g.row] + g.local;
    DH_CHECK(dst + g.cnt <= row_ptr[g.row + 1]);
    for (int t = lane; t < g.cnt; t += 32) { col[dst + t] = acol[g.off + t]; val[dst + t] = aval[g.off + t]; }
  }
}

// exclusive scan of row counts -> row_ptr (single CTA, sequential over chunks; |S| < 2^31 so this is a few ms at most)
__global__ void scan_rows_kernel(const int* __restrict__ cnt, int64_t nd, int64_t* __restrict__ row_ptr) {
  __shared__ int64_t warp_tot[32];
  __shared__ int64_t carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int64_t base = 0; base < nd; base += blockDim.x) {
    int64_t t = base + threadIdx.x;
    int64_t v = t < nd ? cnt[t] : 0, x = v;
    for (int o = 1; o < 32; o <<= 1) { int64_t y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
    if (lane == 31) warp_tot[warp] = x;
    __syncthreads();
    if (warp == 0) {
      int64_t w = lane < (blockDim.x >> 5) ? warp_tot[lane] : 0, s = w;
      for (int o = 1; o < 32; o <<= 1) { int64_t y = __shfl_up_sync(0xffffffffu, s, o); if (lane >= o) s += y; }
      warp_tot[lane] = s - w;
    }
    __syncthreads();
    int64_t excl = carry + warp_tot[warp] + x - v;
    if (t < nd) row_ptr[t] = excl;
    __syncthreads();
    if (threadIdx.x == blockDim.x - 1) carry = excl + v;
    __syncthreads();
  }
  if (threadIdx.x == 0) row_ptr[nd] = carry;
}

// ---------------------------------------------------------------- per-row column sort
// Bitonic network with ascending comparators only (virtual +inf padding stays at the tail).
template <class Sync>
__device__ __forceinline__ void bitonic_rows(int* c, double* v, int len, int tid, int nthr, Sync sync) {
  int N = 2;
  while (N < len) N <<= 1;
  for (int k = 2; k <= N; k <<= 1)
    for (int jj = k >> 1; jj > 0; jj >>= 1) {
      for (int t = tid; t < N / 2; t += nthr) {
        int blk = t / jj, off = t % jj, lo, hi;
        if (jj == (k >> 1)) { lo = blk * k + off; hi = blk * k + k - 1 - off; }
        else { lo = blk * 2 * jj + off; hi = lo + jj; }
        if (hi < len) {
          int cl = c[lo], ch = c[hi];
          if (ch < cl) { double vl = v[lo], vh = v[hi]; c[lo] = ch; c[hi] = cl; v[lo] = vh; v[hi] = vl; }
        }
      }
      sync();
    }
}

constexpr int kSortWarpCap = 512;
__global__ void __launch_bounds__(kWarpsPerCta * 32)
sort_rows_warp_kernel(const int64_t* __restrict__ row_ptr, int64_t nd, int* __restrict__ col, double* __restrict__ val) {
  __shared__ int sc[kWarpsPerCta][kSortWarpCap];
  __shared__ double sv[kWarpsPerCta][kSortWarpCap];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  int64_t row = (int64_t)blockIdx.x * kWarpsPerCta + warp;
  if (row >= nd) return;
  int64_t b = row_ptr[row];
  int len = (int)(row_ptr[row + 1] - b);
  if (len <= 1 || len > kSortWarpCap) return;
  for (int t = lane; t < len; t += 32) { sc[warp][t] = col[b + t]; sv[warp][t] = val[b + t]; }
  __syncwarp();
  bitonic_rows(sc[warp], sv[warp], len, lane, 32, [] { __syncwarp(); });
  for (int t = lane; t < len; t += 32) { col[b + t] = sc[warp][t]; val[b + t] = sv[warp][t]; }
}

// rows longer than kSortWarpCap: one CTA per row.  Chunks of up to kSortCtaCap entries are sorted in shared memory (12 bytes
// per entry; the network's virtual +inf tail pads to a power of two); a longer row is then merged pairwise, run width
// doubling per round: every entry finds its rank in the partner run by a binary search (columns are unique within a row),
// ping-ponging between the CSR and the build arena, which is free once the segments have been copied.
constexpr int kSortCtaCap = 16384;
__global__ void __launch_bounds__(1024)
sort_rows_cta_kernel(const int64_t* __restrict__ row_ptr, int64_t nd, int* __restrict__ col, double* __restrict__ val,
                     int* __restrict__ tcol, double* __restrict__ tval) {
  extern __shared__ __align__(16) unsigned char sort_smem[];
  double* sv = reinterpret_cast<double*>(sort_smem);             // [kSortCtaCap]
  int* sc = reinterpret_cast<int*>(sv + kSortCtaCap);            // [kSortCtaCap]
  for (int64_t row = blockIdx.x; row < nd; row += gridDim.x) {
    const int64_t b = row_ptr[row];
    const int len = (int)(row_ptr[row + 1] - b);
    if (len <= kSortWarpCap) continue;
    for (int c0 = 0; c0 < len; c0 += kSortCtaCap) {
      const int m = min(kSortCtaCap, len - c0);
      for (int t = threadIdx.x; t < m; t += blockDim.x) { sc[t] = col[b + c0 + t]; sv[t] = val[b + c0 + t]; }
      __syncthreads();
      bitonic_rows(sc, sv, m, threadIdx.x, blockDim.x, [] { __syncthreads(); });
      for (int t = threadIdx.x; t < m; t += blockDim.x) { col[b + c0 + t] = sc[t]; val[b + c0 + t] = sv[t]; }
      __syncthreads();
    }
    int* scol = col + b; double* sval = val + b;                 // source of the current merge round
    int* dcol = tcol + b; double* dval = tval + b;
    for (int width = kSortCtaCap; width < len; width <<= 1) {
      for (int t = threadIdx.x; t < len; t += blockDim.x) {
        const int pair0 = (t / (2 * width)) * (2 * width);       // start of this entry's pair of runs
        const int mid = min(pair0 + width, len), end = min(pair0 + 2 * width, len);
        const bool left = t < mid;
        const int key = scol[t];
        int lo = left ? mid : pair0, hi = left ? end : mid;      // the partner run
        while (lo < hi) { const int md = (lo + hi) >> 1; if (scol[md] < key) lo = md + 1; else hi = md; }
        const int pos = left ? t + (lo - mid) : (t - mid) + lo;  // own rank + entries of the partner run below the key
        dcol[pos] = key; dval[pos] = sval[t];
      }
      __syncthreads();
      int* xc = scol; scol = dcol; dcol = xc;
      double* xv = sval; sval = dval; dval = xv;
    }
    if (scol != col + b) {
      for (int t = threadIdx.x; t < len; t += blockDim.x) { col[b + t] = scol[t]; val[b + t] = sval[t]; }
      __syncthreads();
    }
  }
}

template <class K>
dh_status set_smem(detham_ctx* c, K kernel, size_t bytes) {
  DH_CUDA(c, cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
  return DH_OK;
}

}  // namespace

dh_status dh_validate_subspace(detham_ctx* c, const u64* dets, int64_t nd) {
  int* flags = reinterpret_cast<int*>(c->dcount);
  DH_CUDA(c, cudaMemsetAsync(flags, 0, 2 * sizeof(int), c->stream));
  validate_kernel<<<(unsigned)((nd + 255) / 256), 256, 0, c->stream>>>(dets, nd, c->n, c->na, c->nb, flags);
  DH_CUDA(c, cudaGetLastError());
  int* h = reinterpret_cast<int*>(c->pinned);
  DH_CUDA(c, cudaMemcpyAsync(h, flags, 2 * sizeof(int), cudaMemcpyDeviceToHost, c->stream));
  DH_CUDA(c, cudaStreamSynchronize(c->stream));
  if (h[1]) return DH_EPOPCOUNT;
  if (h[0]) return DH_EUNSORTED;
  return DH_OK;
}

dh_status dh_build_shash(detham_ctx* c) {
  int64_t cap = 1024;
  while (cap < 2 * c->nd) cap <<= 1;
  if (cap != c->shash_cap) {
    if (c->shash_key) cudaFree(c->shash_key);
    if (c->shash_idx) cudaFree(c->shash_idx);
    c->shash_key = nullptr; c->shash_idx = nullptr; c->shash_cap = 0;
    DH_CUDA(c, cudaMalloc(&c->shash_key, cap * 2 * sizeof(u64)));
    DH_CUDA(c, cudaMalloc(&c->shash_idx, cap * sizeof(int)));
    c->shash_cap = cap;
  }
  int64_t nbits = 1 << 16;  // >= 64 bits per determinant: 0.1-0.2 % of the non-members pass the filter
  while (nbits < 64 * c->nd && nbits < (1ll << 28)) nbits <<= 1;
  if (nbits != c->sbits_n) {
    if (c->sbits) cudaFree(c->sbits);
    c->sbits = nullptr; c->sbits_n = 0;
    DH_CUDA(c, cudaMalloc(&c->sbits, nbits / 8));
    c->sbits_n = nbits;
  }
  DH_CUDA(c, cudaMemsetAsync(c->sbits, 0, nbits / 8, c->stream));
  DH_CUDA(c, cudaMemsetAsync(c->shash_key, 0, cap * 2 * sizeof(u64), c->stream));
  shash_insert_kernel<<<(unsigned)((c->nd + 255) / 256), 256, 0, c->stream>>>(c->dets, c->nd, c->shash_key, c->shash_idx, (u64)cap,
                                                                            c->sbits, (u64)nbits);
  DH_CUDA(c, cudaGetLastError());
  return DH_OK;
}

static EnumParams make_params(detham_ctx* c, const HbLists* L) {
  EnumParams P;
  P.n = c->n; P.na = c->na; P.nb = c->nb; P.pbits = L->pbits; P.nss = c->n * (c->n - 1) / 2;
  P.h1 = c->h1; P.eri = c->eri; P.sub_off = L->sub_off; P.lval = L->val; P.lab = L->ab; P.lstat = L->stat;
  P.J = c->J; P.JK = c->JK; P.hd = c->hd; P.e_core = c->e_core;
  return P;
}
EnumParams dh_make_params(detham_ctx* c, const HbLists* L) { return make_params(c, L); }

// The CSR a build writes and the index its candidates are looked up in: H_SS (columns = positions in S) or H_SP (row f3:
// columns = positions in the caller's sorted P).  Both share the arena and the row-count buffer.
struct CsrTarget {
  int64_t** row_ptr; int** col; double** val; int64_t* nnz; int64_t* csr_cap; int64_t* row_cap;
  const u64* hkeys; const int* hidx; int64_t hcap; const unsigned* hbits; int64_t hnbits;
};

static dh_status build_csr(detham_ctx* c, const CsrTarget& T, const double* psi /* NULL: H_SS */, double eps) {
  const bool sp = psi != nullptr;
  const HbLists* L = nullptr;
  dh_status st = dh_get_lists(c, 0, &L);
  if (st != DH_OK) return st;
  EnumParams P = make_params(c, L);
  const int64_t nd = c->nd;
  if (c->row_cnt_cap < nd) {
    if (c->row_cnt) cudaFree(c->row_cnt);
    c->row_cnt = nullptr; c->row_cnt_cap = 0;
    DH_CUDA(c, cudaMalloc(&c->row_cnt, nd * sizeof(int)));
    c->row_cnt_cap = nd;
  }
  if (*T.row_cap < nd) {
    if (*T.row_ptr) cudaFree(*T.row_ptr);
    *T.row_ptr = nullptr; *T.row_cap = 0;
    DH_CUDA(c, cudaMalloc(T.row_ptr, (nd + 1) * sizeof(int64_t)));
    *T.row_cap = nd;
  }
  *T.nnz = -1;
  const size_t smem = ((dh_cta_table_bytes(c->n) + 15) & ~(size_t)15) + kBuildWarps * sizeof(WarpScratch);
  st = sp ? set_smem(c, build_kernel<true>, smem) : set_smem(c, build_kernel<false>, smem);
  if (st != DH_OK) return st;
  int64_t want = (nd + kBuildWarps - 1) / kBuildWarps;
  const int grid = (int)(want < (int64_t)c->sm_count * 2 ? want : (int64_t)c->sm_count * 2);
  const int64_t slack = (int64_t)grid * kBuildWarps * kBlk;  // every warp may leave one block partly used
  int* overflow = reinterpret_cast<int*>(c->dcount + 8);
  int64_t* h = reinterpret_cast<int64_t*>(c->pinned);
  int64_t nnz = 0;
  double ms_pass = 0.0;
  int64_t want_arena = c->arena_cap > 0 ? c->arena_cap : nd * 64 + slack;  // first build: a guess; later: the last size
  for (int attempt = 0;; ++attempt) {
    if (c->arena_cap < want_arena) {
      if (c->acol) cudaFree(c->acol);
      if (c->aval) cudaFree(c->aval);
      c->acol = nullptr; c->aval = nullptr; c->arena_cap = 0;
      DH_CUDA(c, cudaMalloc(&c->acol, want_arena * sizeof(int)));
      DH_CUDA(c, cudaMalloc(&c->aval, want_arena * sizeof(double)));
      c->arena_cap = want_arena;
    }
    // segments: at least one per non-empty row plus one per arena block; sized on its own, because a context reused for a
    // larger subspace (the outer loop of Alg. 1) can need more rows than the arena of an earlier build implies
    const int64_t need_seg = nd + c->arena_cap / kBlk + 4096;
    if (c->seg_cap < need_seg) {
      if (c->segs) cudaFree(c->segs);
      c->segs = nullptr; c->seg_cap = 0;
      DH_CUDA(c, cudaMalloc(&c->segs, need_seg * sizeof(Seg)));
      c->seg_cap = need_seg;
    }
    DH_CUDA(c, cudaMemsetAsync(c->dcount, 0, 16 * sizeof(u64), c->stream));
    DH_TICK(c, 0);
    auto kernel = sp ? build_kernel<true> : build_kernel<false>;
    kernel<<<grid, kBuildWarps * 32, smem, c->stream>>>(P, c->dets, psi, nd, eps, T.hkeys, T.hidx, (u64)T.hcap, T.hbits, (u64)T.hnbits,
                                                        c->row_cnt, c->acol, c->aval, c->arena_cap,
                                                        reinterpret_cast<Seg*>(c->segs), c->seg_cap, c->dcount, overflow);
    DH_CUDA(c, cudaGetLastError());
    scan_rows_kernel<<<1, 1024, 0, c->stream>>>(c->row_cnt, nd, *T.row_ptr);
    DH_CUDA(c, cudaGetLastError());
    DH_TICK(c, 1);
    DH_CUDA(c, cudaMemcpyAsync(h, *T.row_ptr + nd, sizeof(int64_t), cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(c, cudaMemcpyAsync(h + 1, c->dcount, 4 * sizeof(u64), cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(c, cudaMemcpyAsync(h + 5, overflow, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(c, cudaStreamSynchronize(c->stream));
    ms_pass += dh_elapsed(c, 0, 1);
    nnz = h[0];
    if (sp) c->ctr.hsp_generated = h[2]; else c->ctr.build_generated = h[2];
    if (!*reinterpret_cast<int*>(h + 5)) break;
    if (attempt >= 1) return DH_ENOMEM;  // cannot happen: the second attempt is sized from the exact count
    want_arena = nnz + nnz / 32 + slack;  // a block is closed when the next batch of <= 32 hits does not fit: < 32 of 1024 entries lost
  }
  const int64_t nseg = h[4];
  if (*T.csr_cap < nnz) {
    if (*T.col) cudaFree(*T.col);
    if (*T.val) cudaFree(*T.val);
    *T.col = nullptr; *T.val = nullptr; *T.csr_cap = 0;
    const int64_t cap = nnz > 0 ? nnz : 1;
    DH_CUDA(c, cudaMalloc(T.col, cap * sizeof(int)));
    DH_CUDA(c, cudaMalloc(T.val, cap * sizeof(double)));
    *T.csr_cap = cap;
  }
  DH_TICK(c, 2);
  {
    int64_t blocks = (nseg + 7) / 8;
    const int cgrid = (int)(blocks < (int64_t)c->sm_count * 8 ? (blocks > 0 ? blocks : 1) : (int64_t)c->sm_count * 8);
    copy_segs_kernel<<<cgrid, 256, 0, c->stream>>>(reinterpret_cast<const Seg*>(c->segs), nseg, *T.row_ptr, c->acol, c->aval, *T.col, *T.val);
    DH_CUDA(c, cudaGetLastError());
  }
  sort_rows_warp_kernel<<<(unsigned)((nd + kWarpsPerCta - 1) / kWarpsPerCta), kWarpsPerCta * 32, 0, c->stream>>>(*T.row_ptr, nd, *T.col, *T.val);
  DH_CUDA(c, cudaGetLastError());
  {
    const size_t sort_smem = (size_t)kSortCtaCap * (sizeof(double) + sizeof(int));
    st = set_smem(c, sort_rows_cta_kernel, sort_smem); if (st != DH_OK) return st;
    sort_rows_cta_kernel<<<c->sm_count, 1024, sort_smem, c->stream>>>(*T.row_ptr, nd, *T.col, *T.val, c->acol, c->aval);
  }
  DH_CUDA(c, cudaGetLastError());
  DH_TICK(c, 3);
  DH_CUDA(c, cudaEventSynchronize(c->ev[3]));
  if (sp) {
    c->ctr.ms_hsp_build = ms_pass;
    c->ctr.ms_hsp_fill = dh_elapsed(c, 2, 3);
    c->ctr.hsp_nnz = nnz;
  } else {
    c->ctr.ms_build_count = ms_pass;
    c->ctr.ms_build_fill = dh_elapsed(c, 2, 3);
    c->ctr.nnz = nnz;
  }
  *T.nnz = nnz;
  return DH_OK;
}

dh_status dh_ham_build(detham_ctx* c, double eps) {
  // Two organisations with identical results.  By excitation degree (pair_build.cu) the cost grows like the number of pairs of
  // determinants whose alpha strings are within a double excitation of each other; walking the heat-bath lists it grows like
  // |S| x (screened excitations per source).  Measured on B200 (profiles/r2_summary.md), list walk against pairs: H2O-shaped
  // |S| = 2e4 3.9 / 5.6 ms, N2-shaped 1e5 33.7 / 21.2 ms, Cr2-shaped 1e6 1565 / 583 ms (1e5 screened excitations per source,
  // 98 % of them not in S): pairs from 2^16 determinants on.
  const bool pairs = c->build_method == 2 || (c->build_method == 0 && c->nd >= (1ll << 16) && c->nd <= (4ll << 20));
  if (pairs) return dh_pair_build(c, eps);
  c->ctr.build_pairs = 0;
  CsrTarget T{&c->row_ptr, &c->col, &c->val, &c->nnz, &c->csr_cap, &c->row_cap,
              c->shash_key, c->shash_idx, c->shash_cap, c->sbits, c->sbits_n};
  return build_csr(c, T, nullptr, eps);
}

// H_SP (row f3; "constructs the sparse Hamiltonian blocks H_VV and H_VP in CSR format", Eq. 8 PAPER.md:126,
// Eq. S3): rows = determinants of S, columns = positions in the caller's sorted, deduplicated key list P
// (detham_expand's output or any sorted subset of it), values H_{P_k, i} of the couplings the screen of Eq. 14 generates.
// open-addressing index of the caller's sorted key list P (validated: strictly ascending, electron counts, high bits clear)
static dh_status build_p_index(detham_ctx* c, const u64* pkeys, int64_t m) {
  dh_status st = m > 0 ? dh_validate_subspace(c, pkeys, m) : DH_OK;
  if (st != DH_OK) return st;
  int64_t cap = 1024;
  while (cap < 2 * m) cap <<= 1;
  if (cap != c->phash_cap) {
    if (c->phash_key) cudaFree(c->phash_key);
    if (c->phash_idx) cudaFree(c->phash_idx);
    c->phash_key = nullptr; c->phash_idx = nullptr; c->phash_cap = 0;
    DH_CUDA(c, cudaMalloc(&c->phash_key, cap * 2 * sizeof(u64)));
    DH_CUDA(c, cudaMalloc(&c->phash_idx, cap * sizeof(int)));
    c->phash_cap = cap;
  }
  DH_CUDA(c, cudaMemsetAsync(c->phash_key, 0, cap * 2 * sizeof(u64), c->stream));
  if (m > 0) {
    shash_insert_kernel<<<(unsigned)((m + 255) / 256), 256, 0, c->stream>>>(pkeys, m, c->phash_key, c->phash_idx, (u64)cap, nullptr, 0ull);
    DH_CUDA(c, cudaGetLastError());
  }
  return DH_OK;
}

dh_status dh_hsp_build(detham_ctx* c, const double* psi, double eps2, const u64* pkeys, int64_t m) {
  dh_status st = build_p_index(c, pkeys, m);
  if (st != DH_OK) return st;
  c->sp_cols = m;
  CsrTarget T{&c->sp_row_ptr, &c->sp_col, &c->sp_val, &c->sp_nnz, &c->sp_csr_cap, &c->sp_row_cap,
              c->phash_key, c->phash_idx, c->phash_cap, nullptr, 0};
  return build_csr(c, T, psi, eps2);
}

// The complete-the-sum amplitude (row f2; Eq. 13: <x|H|Psi_V>, the full projection): v_out[k] = sum over ALL i in S of
// H_{P_k, i} psi_i for the caller's sorted key list P.  One unscreened enumeration of every source, looked up in the index of P,
// accumulated with RED.ADD.F64 (the order of the additions varies from run to run).
dh_status dh_complete_sum(detham_ctx* c, const double* psi, const u64* pkeys, int64_t m, double* v_out) {
  dh_status st = build_p_index(c, pkeys, m);
  if (st != DH_OK) return st;
  if (m == 0) return DH_OK;
  const HbLists* L = nullptr;
  st = dh_get_lists(c, 0, &L); if (st != DH_OK) return st;
  EnumParams P = make_params(c, L);
  const size_t smem = ((dh_cta_table_bytes(c->n) + 15) & ~(size_t)15) + kBuildWarps * sizeof(WarpScratch);
  st = set_smem(c, complete_kernel, smem); if (st != DH_OK) return st;
  int64_t want = (c->nd + kBuildWarps - 1) / kBuildWarps;
  const int grid = (int)(want < (int64_t)c->sm_count * 2 ? want : (int64_t)c->sm_count * 2);
  DH_CUDA(c, cudaMemsetAsync(v_out, 0, (size_t)m * sizeof(double), c->stream));
  DH_CUDA(c, cudaMemsetAsync(c->dcount, 0, 16 * sizeof(u64), c->stream));
  complete_kernel<<<grid, kBuildWarps * 32, smem, c->stream>>>(P, c->dets, psi, c->nd, c->phash_key, c->phash_idx, (u64)c->phash_cap, v_out, c->dcount);
  DH_CUDA(c, cudaGetLastError());
  DH_CUDA(c, cudaStreamSynchronize(c->stream));
  return DH_OK;
}
