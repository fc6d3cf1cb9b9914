// Shared declarations of the detham CUDA library (sm_100a only).  Nothing here is used by oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "detham.h"

typedef unsigned long long u64;

#define DH_WARP 32
#define DH_MAX_ORB 64
#define DH_MAX_PBITS 10  // up to 1024 key partitions

// ---------------------------------------------------------------- heat-bath lists
// Three families of segments, one segment per ordered/unordered orbital pair:
//   family 0 (alpha-alpha), 1 (beta-beta): pair i<j, id = j(j-1)/2 + i; entries (a<b), a,b not in {i,j};
//                                          value <ij||ab> = (ia|jb) - (ib|ja)
//   family 2 (alpha-beta): pair (i alpha, j beta), id = i*n + j; entries (a != i, b != j); value (ia|jb)
// Inside a segment the entries are grouped by key-partition class (Zobrist class of the pair (a,b) in that family's
// spins) and, inside a class, sorted by |value| descending (ties: (a,b) ascending).  sub_off[seg * P + c] is the
// start of class c of segment seg; sub_off[nseg * P] = total.
struct HbLists {
  int pbits = -1;            // P = 1 << pbits
  int nseg = 0;
  int64_t total = 0;
  int* sub_off = nullptr;       // device int32 [nseg * P + 1]
  double* val = nullptr;        // device fp64 [total]
  unsigned short* ab = nullptr; // device u16 [total]: a | (b << 8)
  double* stat = nullptr;       // device fp64 [total]: the source-independent part of H_aa - H_ii for the entry's double
                                // excitation, X_ij + X_ab - (J-K)_ia - (J-K)_jb - X_ib - X_ja with X = J-K (same spin) or J
};

struct detham_ctx {
  int n = 0, na = 0, nb = 0;
  double e_core = 0.0;
  cudaStream_t stream = nullptr;
  int device = 0;
  int sm_count = 148;
  std::string cuda_err;

  // integral store (a2): L2-resident
  double* h1 = nullptr;   // [n*n]
  double* eri = nullptr;  // packed
  int64_t n_eri = 0;
  double* J = nullptr;    // [n*n]  (pp|qq)
  double* JK = nullptr;   // [n*n]  (pp|qq) - (pq|qp)
  double* hd = nullptr;   // [n]    h_pp

  HbLists lists[DH_MAX_PBITS + 1];  // built on demand per partition count

  // determinant store (a1)
  const u64* dets = nullptr;  // borrowed, device [nd][2]
  int64_t nd = 0;
  u64* dets_owned = nullptr;  // only for detham_solve_host
  double* psi_owned = nullptr;
  int64_t owned_cap = 0;
  u64* shash_key = nullptr;   // device [shash_cap][2], open addressing, EMPTY = {0,0}
  int* shash_idx = nullptr;   // device [shash_cap]
  int64_t shash_cap = 0;
  unsigned* sbits = nullptr;  // membership pre-filter (dh_maybe_member): sbits_n bits, two set per D in S
  int64_t sbits_n = 0;

  // CSR H_SS (a6)
  int64_t* row_ptr = nullptr;
  int* col = nullptr;
  double* val = nullptr;
  int64_t nnz = -1;
  int64_t csr_cap = 0;
  int64_t row_cap = 0;     // rows row_ptr has room for
  int* row_cnt = nullptr;  // device int32 [nd], shared by the H_SS and H_SP builds
  int64_t row_cnt_cap = 0;
  int* acol = nullptr;     // build arena: hits in warp order, copied to col/val once the row offsets are known
  double* aval = nullptr;
  int64_t arena_cap = 0;   // entries
  void* segs = nullptr;    // arena segments
  int64_t seg_cap = 0;

  // ham_build by excitation degree (pair_build.cu): alpha groups of the sorted S, diagonals
  u64* pair_galpha = nullptr; int64_t pair_group_cap = 0;
  int* pair_gstart = nullptr; int64_t pair_gstart_cap = 0;
  double* pair_diag = nullptr; int64_t pair_diag_cap = 0;
  u64* pair_akey = nullptr; int64_t pair_akey_cap = 0;   // arena tags: row << 32 | place in the row (values in acol / aval)
  int* pair_bused = nullptr; int64_t pair_bused_cap = 0;  // entries used of every arena block
  int build_method = 0;  // detham_build_config: 0 choose, 1 list walk, 2 excitation degree

  // CSR H_SP (row f3) and the lookup index of the caller's P it was built against
  int64_t* sp_row_ptr = nullptr;
  int* sp_col = nullptr;
  double* sp_val = nullptr;
  int64_t sp_nnz = -1;
  int64_t sp_csr_cap = 0;
  int64_t sp_row_cap = 0;
  int64_t sp_cols = 0;
  u64* phash_key = nullptr;
  int* phash_idx = nullptr;
  int64_t phash_cap = 0;

  // pt2
  void* table = nullptr;      // zero between calls (the scan clears what it reads)
  int64_t table_slots = 0;
  std::vector<double> partials;
  void* pool = nullptr;       // streamed PT2: contribution records {key, H psi, H_aa} of one pass, [bin][CTA][seg_cap]
  int64_t pool_bytes = 0;
  void* ring = nullptr;       // streamed PT2: the L2-resident region tables
  size_t ring_bytes = 0;
  void* sflags = nullptr;     // streamed PT2: records per (bin, CTA) segment + the hand-over counters of the merge
  size_t sflags_bytes = 0;
  std::vector<cudaEvent_t> sev;  // per-pass timers of the streamed PT2
  detham_pt2_options opt{};   // detham_pt2_set_options (zero = defaults)
  bool debug = false;         // DETHAM_DEBUG=1 at detham_create: planning decisions go to stderr

  // scratch
  double* red = nullptr;      // device reduction buffer
  int64_t red_cap = 0;
  u64* dcount = nullptr;      // device counters [64]
  int* perm = nullptr;        // pt2: sources in key-class order
  int64_t perm_cap = 0;
  void* scratch = nullptr;    // grow-only work space of ediag / expand / connections (dh_scratch), freed by detham_trim
  size_t scratch_bytes = 0;
  void* pinned = nullptr;     // pinned host scratch (4 KB)
  int64_t* hist = nullptr;    // device int64 [1024] class histogram

  detham_counters ctr{};
  cudaEvent_t ev[8] = {};  // scratch events for the per-phase timers
};

// record ev[k] on the context's stream
#define DH_TICK(ctx, k) DH_CUDA(ctx, cudaEventRecord((ctx)->ev[k], (ctx)->stream))
inline double dh_elapsed(detham_ctx* c, int a, int b) { float ms = 0.f; cudaEventElapsedTime(&ms, c->ev[a], c->ev[b]); return (double)ms; }

#define DH_CUDA(ctx, expr)                                                     \
  do {                                                                         \
    cudaError_t _e = (expr);                                                   \
    if (_e != cudaSuccess) {                                                   \
      (ctx)->cuda_err = std::string(#expr) + ": " + cudaGetErrorString(_e);    \
      return _e == cudaErrorMemoryAllocation ? DH_ENOMEM : DH_ECUDA;           \
    }                                                                          \
  } while (0)

// entry points implemented across the translation units
dh_status dh_build_jk(detham_ctx* c);
dh_status dh_get_lists(detham_ctx* c, int pbits, const HbLists** out);
dh_status dh_ham_build(detham_ctx* c, double eps);
dh_status dh_pair_build(detham_ctx* c, double eps);
dh_status dh_hsp_build(detham_ctx* c, const double* psi, double eps2, const u64* pkeys, int64_t m);
dh_status dh_complete_sum(detham_ctx* c, const double* psi, const u64* pkeys, int64_t m, double* v_out);
dh_status dh_energy(detham_ctx* c, const double* psi, double* e_out, double* n2_out, double* y_out);
dh_status dh_expand(detham_ctx* c, const double* psi, double eps2, u64* keys_out, double* score_out, double* v_out, double* haa_out,
                    int64_t cap, int64_t* n_out);
dh_status dh_ediag(detham_ctx* c, const double* v0, double tol, int max_iter, double* e_out, int* iters_out, double* resid_out,
                   int* converged_out);
dh_status dh_residual(detham_ctx* c, const double* psi, double e_s, double* r_out, double* internal_out);
dh_status dh_pt2(detham_ctx* c, const double* psi, double e_s, double eps2, double* out);
dh_status dh_count_screened(detham_ctx* c, const double* psi, double thr, int64_t* n_out);
dh_status dh_connections(detham_ctx* c, int64_t row, double tau, std::vector<u64>& keys, std::vector<double>& h);
dh_status dh_diagonals(detham_ctx* c, const u64* dets, int64_t m, double* out);
dh_status dh_build_shash(detham_ctx* c);
dh_status dh_validate_subspace(detham_ctx* c, const u64* dets, int64_t nd);
dh_status dh_ensure_red(detham_ctx* c, int64_t n);
// the context's work space, at least `bytes` long and 256-byte aligned; contents do not survive a call that asks for more
dh_status dh_scratch(detham_ctx* c, size_t bytes, void** p);

// ---------------------------------------------------------------- device helpers
#ifdef __CUDACC__

__host__ __device__ __forceinline__ int dh_tri(int x, int y) { return x >= y ? x * (x + 1) / 2 + y : y * (y + 1) / 2 + x; }

// chemist (pq|rs) from the packed 8-fold array
__device__ __forceinline__ double dh_eri(const double* __restrict__ eri, int p, int q, int r, int s) {
  int pq = dh_tri(p, q), rs = dh_tri(r, s);
  return __ldg(eri + (pq >= rs ? pq * (pq + 1) / 2 + rs : rs * (rs + 1) / 2 + pq));
}

// Key-partition words (reading Q14): word of spin-orbital index s (alpha p -> p, beta q -> 64 + q) is
// splitmix64(260121310 + s); a determinant's word is the XOR over its occupied spin-orbitals.
__host__ __device__ __forceinline__ u64 dh_zword(int s) {
  u64 x = 260121310ull + (u64)s + 0x9E3779B97F4A7C15ull;
  x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
  x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
  return x ^ (x >> 31);
}

struct __align__(16) Key128 { u64 a, b; };

__device__ __forceinline__ Key128 dh_cas128(void* addr, Key128 cmp, Key128 val) {
  Key128 old;
  asm volatile(
      "{\n\t.reg .b128 c, v, o;\n\t"
      "mov.b128 c, {%2, %3};\n\t"
      "mov.b128 v, {%4, %5};\n\t"
      "atom.relaxed.gpu.global.cas.b128 o, [%6], c, v;\n\t"
      "mov.b128 {%0, %1}, o;\n\t}"
      : "=l"(old.a), "=l"(old.b)
      : "l"(cmp.a), "l"(cmp.b), "l"(val.a), "l"(val.b), "l"(addr)
      : "memory");
  return old;
}

// one 32-byte slot in one transaction (LDG.E.256), coherent at gpu scope (bypasses the non-coherent L1)
__device__ __forceinline__ void dh_ld256(const void* p, u64& a, u64& b, u64& c, u64& d) {
  asm volatile("ld.relaxed.gpu.global.v4.u64 {%0,%1,%2,%3}, [%4];" : "=l"(a), "=l"(b), "=l"(c), "=l"(d) : "l"(p) : "memory");
}

// streaming variants for the table scan (evict-first: the scan touches every slot exactly once)
__device__ __forceinline__ void dh_ld256_cs(const void* p, u64& a, u64& b, u64& c, u64& d) {
  asm volatile("ld.global.cs.v4.u64 {%0,%1,%2,%3}, [%4];" : "=l"(a), "=l"(b), "=l"(c), "=l"(d) : "l"(p) : "memory");
}
__device__ __forceinline__ void dh_st256(void* p, u64 a, u64 b, u64 c, u64 d) {
  asm volatile("st.global.v4.u64 [%0], {%1,%2,%3,%4};" ::"l"(p), "l"(a), "l"(b), "l"(c), "l"(d) : "memory");
}
__device__ __forceinline__ void dh_st256_zero(void* p) {
  asm volatile("st.global.cs.v4.u64 [%0], {%1,%1,%1,%1};" ::"l"(p), "l"(0ull) : "memory");
}

// (-1)^(electrons of word w strictly between orbitals x and y): returns 0 (even) or 1 (odd)
__device__ __forceinline__ int dh_parity_between(u64 w, int x, int y) {
  int lo = min(x, y), hi = max(x, y);
  u64 m = ((1ull << hi) - 1ull) & ~((2ull << lo) - 1ull);
  return __popcll(w & m) & 1;
}

// lookup in the L2-resident open-addressing index of S (built by shash_insert_kernel): index of (ka, kb) or -1
__device__ __forceinline__ int dh_shash_find(const u64* __restrict__ keys, const int* __restrict__ idx, u64 cap, u64 ka, u64 kb, u64 z) {
  u64 slot = __umul64hi(z, cap);
  for (;;) {
    ulonglong2 k = __ldg(reinterpret_cast<const ulonglong2*>(keys) + slot);
    if (k.x == ka && k.y == kb) return __ldg(idx + slot);
    if (k.x == 0ull && k.y == 0ull) return -1;
    if (++slot == cap) slot = 0;
  }
}

// membership pre-filter of the determinant store: false = certainly not in S (one 8-byte L2 load).  A blocked Bloom filter:
// `nbits` (a power of two, >= 64 per determinant) bits seen as 64-bit words; a determinant sets two bits of the word its
// partition word selects.  About 0.1-0.2 % of the non-members pass, so a warp of candidates rarely diverges into the index.
// Bounds checks of the checked build (libdetham_checked.so, -DDETHAM_CHECKED; paper_2601_21310_b200/build.py): device asserts at
// every computed index into a queue, arena, pool, table or output array.  compute-sanitizer is not available on the GPU pool
// this was developed on; tests/test_gpu_parity.py::test_checked_build runs the small cases through this build instead.
#ifdef DETHAM_CHECKED
#include <assert.h>
#define DH_CHECK(cond) assert(cond)
#else
#define DH_CHECK(cond) ((void)0)
#endif

__device__ __forceinline__ u64 dh_filter_mask(u64 z) { return (1ull << ((z >> 10) & 63ull)) | (1ull << ((z >> 16) & 63ull)); }
__device__ __forceinline__ u64 dh_filter_word(u64 nbits, u64 z) { return z >> (__clzll((long long)nbits) + 7); }
__device__ __forceinline__ bool dh_maybe_member(const unsigned* __restrict__ bits, u64 nbits, u64 z) {
  const u64 m = dh_filter_mask(z);
  return (__ldg(reinterpret_cast<const u64*>(bits) + dh_filter_word(nbits, z)) & m) == m;
}

#endif  // __CUDACC__
