// ham_build by excitation degree (a6, second organisation): instead of enumerating the ~1e5 screened excitations of every
// source and looking each up in S (98 % are not there on the Cr2-shaped config), find the pairs (D_i, D_j) of S that differ
// by at most a double excitation directly and evaluate the Slater-Condon element (a5) of those only.
//
// S is sorted by (alpha, beta), so determinants with the same alpha string are contiguous ("alpha groups").  Two
// determinants are connected iff popc(alpha_i ^ alpha_j) + popc(beta_i ^ beta_j) <= 4.  A warp owns 32 consecutive rows; it
// tests the alpha strings of its rows (a handful of distinct ones) against every group's alpha string, 32 groups per step,
// and for the group pairs within reach walks the group's beta strings 32 at a time.  Rows come out in column order (groups
// ascending, members ascending), so the CSR needs no sort; one counting pass sizes it, a second pass fills it.
//
// Values are the very expressions of the list walker (lists.cu, enumerate.cuh) - one packed integral or the difference of two
// for doubles, the ordered sum of reading Q7 for singles - so both organisations give the same bits.
#include <algorithm>

#include "pt2_common.cuh"

EnumParams dh_make_params(detham_ctx* c, const HbLists* L);

namespace {

constexpr int kPairWarps = 8;
constexpr int kArenaBlk = 1024;  // arena entries a warp reserves at a time

__global__ void group_flag_kernel(const u64* __restrict__ dets, int64_t nd, int* __restrict__ flag) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t < nd) flag[t] = (t == 0 || dets[2 * t] != dets[2 * (t - 1)]) ? 1 : 0;
}

// exclusive prefix sum of n ints into int64 out[n + 1] (one CTA; n up to a few 1e7 is a millisecond or two)
__global__ void __launch_bounds__(1024) excl_scan_kernel(const int* __restrict__ in, int64_t n, int64_t* __restrict__ out) {
  __shared__ int64_t part[1024];
  const int t = threadIdx.x;
  const int64_t per = (n + 1023) / 1024, b = t * per, e = b + per < n ? b + per : n;
  int64_t s = 0;
  for (int64_t k = b; k < e; ++k) s += in[k];
  part[t] = s;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {
    int64_t v = t >= o ? part[t - o] : 0;
    __syncthreads();
    part[t] += v;
    __syncthreads();
  }
  int64_t run = part[t] - s;
  for (int64_t k = b; k < e; ++k) { out[k] = run; run += in[k]; }
  if (t == 1023) out[n] = part[1023];
}

__global__ void group_fill_kernel(const u64* __restrict__ dets, int64_t nd, const int* __restrict__ flag, const int64_t* __restrict__ pre,
                                  u64* __restrict__ galpha, int* __restrict__ gstart) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t < nd && flag[t]) { galpha[pre[t]] = dets[2 * t]; gstart[pre[t]] = (int)t; }
  if (t == nd) gstart[pre[nd]] = (int)nd;
}

__global__ void pair_diag_kernel(int n, const double* __restrict__ J, const double* __restrict__ JK, const double* __restrict__ hd,
                                 double e_core, const u64* __restrict__ dets, int64_t m, double* __restrict__ out) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t < m) out[t] = dh_diag_from_scratch(n, J, JK, hd, e_core, dets[2 * t], dets[2 * t + 1]);
}

// position in [js, je) of the determinant with beta string `b` (the determinants of an alpha group are sorted by beta), or -1
__device__ __forceinline__ int dh_find_beta(const u64* __restrict__ dets, int js, int je, u64 b) {
  int lo = js, hi = je;
  while (hi - lo > 1) {  // invariant: beta[lo] <= b if it is there at all
    const int mid = (lo + hi) >> 1;
    if (__ldg(dets + 2 * (int64_t)mid + 1) <= b) lo = mid; else hi = mid;
  }
  return (lo < je && __ldg(dets + 2 * (int64_t)lo + 1) == b) ? lo : -1;
}

// Single-excitation element i -> a in the spin string `ws` of the SOURCE (the other string is `wo`): the ordered sum of reading
// Q7 - h_ia, then ((ia|qq) - (iq|qa)) over same-spin occupied q ascending, then (ia|qq) over other-spin occupied q ascending -
// exactly dh_single_value_occ's additions, with the occupied orbitals taken from the words instead of a list.
__device__ double pair_single_value(const EnumParams& P, u64 ws, u64 wo, int i, int a) {
  double v = __ldg(P.h1 + i * P.n + a);
  for (u64 m = ws; m;) { const int q = __ffsll((long long)m) - 1; m &= m - 1; v = v + (dh_eri(P.eri, i, a, q, q) - dh_eri(P.eri, i, q, q, a)); }
  for (u64 m = wo; m;) { const int q = __ffsll((long long)m) - 1; m &= m - 1; v = v + dh_eri(P.eri, i, a, q, q); }
  return dh_parity_between(ws, i, a) ? -v : v;
}

// <D_j|H|D_r> for D_j a single or double excitation of the source D_r = (ar, br)  (xa, xb: the XOR of the strings)
__device__ double pair_element(const EnumParams& P, u64 ar, u64 br, u64 xa, u64 xb) {
  const int ea = __popcll(xa) >> 1, eb = __popcll(xb) >> 1;
  if (ea + eb == 1) {
    const int s = eb;  // 0: alpha single, 1: beta single
    const u64 w = s ? br : ar, x = s ? xb : xa;
    const int i = __ffsll((long long)(x & w)) - 1, a = __ffsll((long long)(x & ~w)) - 1;
    return pair_single_value(P, w, s ? ar : br, i, a);
  }
  if (ea == 1) {  // alpha-beta double: (ia|jb), phase = product of the two single phases (reading Q1)
    const int i = __ffsll((long long)(xa & ar)) - 1, a = __ffsll((long long)(xa & ~ar)) - 1;
    const int j = __ffsll((long long)(xb & br)) - 1, b = __ffsll((long long)(xb & ~br)) - 1;
    const double v = dh_eri(P.eri, i, a, j, b);
    return dh_double_parity(ar, br, 2, 0, i, j, a, b) ? -v : v;
  }
  const int s = eb ? 1 : 0;  // same-spin double i<j -> a<b: <ij||ab> = (ia|jb) - (ib|ja)
  const u64 w = s ? br : ar, x = s ? xb : xa;
  u64 h = x & w, q = x & ~w;
  const int i = __ffsll((long long)h) - 1; h &= h - 1;
  const int j = __ffsll((long long)h) - 1;
  const int a = __ffsll((long long)q) - 1; q &= q - 1;
  const int b = __ffsll((long long)q) - 1;
  const double v = dh_eri(P.eri, i, a, j, b) - dh_eri(P.eri, i, b, j, a);
  return dh_double_parity(ar, br, 1, s, i, j, a, b) ? -v : v;
}

// One pass: every kept entry goes to an arena (blocks of kArenaBlk entries per warp) tagged with its row and its place in the row,
// and the rows are counted; after the row scan a scatter moves the entries to their CSR positions.  If the arena is too small the
// pass still counts exactly and is run again with the exact size.
// Pairs within reach are queued per warp as (row of the block, column) in the order they are found and evaluated 32 at a time,
// so that the Slater-Condon evaluation (a few hundred instructions, two to ~40 integral loads) runs with every lane busy; an
// entry's place in its row is the row's running count plus its rank among the batch's kept entries of the same row.
__global__ void __launch_bounds__(kPairWarps * 32)
pair_kernel(EnumParams P, const u64* __restrict__ dets, int64_t nd, double eps, const u64* __restrict__ galpha,
            const int* __restrict__ gstart, int ngroups, const double* __restrict__ diag, int* __restrict__ row_cnt,
            u64* __restrict__ akey, int* __restrict__ acol, double* __restrict__ aval, int* __restrict__ bused, int64_t arena_cap,
            u64* counters /* [0] next block of rows [1] elements evaluated [2] arena cursor */, int* overflow) {
  __shared__ int s_qcol[kPairWarps][64];
  __shared__ unsigned char s_qrow[kPairWarps][64];
  __shared__ int s_cnt[kPairWarps][32];
  __shared__ int s_tg[kPairWarps][64];            // pending look-ups: alpha group ...
  __shared__ unsigned char s_tr[kPairWarps][64];  // ... and row of the block whose beta string is looked up in it
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned full = 0xffffffffu, lt = (1u << lane) - 1u;
  int* qcol = s_qcol[warp];
  unsigned char* qrow = s_qrow[warp];
  int* cnt = s_cnt[warp];
  int* tg = s_tg[warp];
  unsigned char* tr = s_tr[warp];
  u64 evaluated = 0;
  int64_t wpos = 0, wend = 0;  // this warp's window in the arena (wpos < 0: arena exhausted, count only)
  for (;;) {
    u64 blk = 0;
    if (lane == 0) blk = atomicAdd(counters, 1ull);
    blk = __shfl_sync(full, blk, 0);
    const int64_t row0 = (int64_t)blk * 32;
    if (row0 >= nd) break;
    const int64_t row = row0 + lane;
    const bool have = row < nd;
    const u64 ar = have ? dets[2 * row] : 0ull, br = have ? dets[2 * row + 1] : 0ull;
    cnt[lane] = 0;
    int qn = 0;
    __syncwarp();
    // evaluate the first `take` queued pairs (all lanes take part in the shuffles), then close the queue up
    auto flush = [&](int take) {
      const bool mine = lane < take;
      const int r = mine ? (int)qrow[lane] : 0;
      const int j = mine ? qcol[lane] : 0;
      const u64 a_row = __shfl_sync(full, ar, r), b_row = __shfl_sync(full, br, r);
      bool keep = false;
      double v = 0.0;
      if (mine) {
        const ulonglong2 dj = __ldg(reinterpret_cast<const ulonglong2*>(dets) + j);
        const u64 xa = a_row ^ dj.x, xb = b_row ^ dj.y;
        if ((xa | xb) == 0ull) { v = diag[j]; keep = true; }  // the row's own determinant: the diagonal is always stored (reading Q4)
        else {
          v = pair_element(P, a_row, b_row, xa, xb);
          ++evaluated;
          keep = v != 0.0 && fabs(v) >= eps;
        }
      }
      const unsigned peers = __match_any_sync(full, keep ? r : 64 + lane);  // kept entries of the same row
      const unsigned km = __ballot_sync(full, keep);
      if (km) {  // warp-uniform: room in the arena for this batch
        const int nk = __popc(km);
        if (wpos >= 0 && wpos + nk > wend) {
          if (lane == 0 && wend > 0) bused[(wend - 1) / kArenaBlk] = (int)(wpos - (wend - kArenaBlk));
          u64 nb = 0;
          if (lane == 0) nb = atomicAdd(counters + 2, (u64)kArenaBlk);
          nb = __shfl_sync(full, nb, 0);
          if ((int64_t)nb + kArenaBlk > arena_cap) { wpos = -1; if (lane == 0) *overflow = 1; }
          else { wpos = (int64_t)nb; wend = wpos + kArenaBlk; }
        }
      }
      if (keep) {
        const int at = cnt[r];
        const int k = at + __popc(peers & lt);
        if (wpos >= 0) {
          const int64_t e = wpos + __popc(km & lt);
          DH_CHECK(e >= 0 && e < arena_cap && j >= 0 && j < nd);
          akey[e] = ((u64)(unsigned)(row0 + r) << 32) | (u64)(unsigned)k; acol[e] = j; aval[e] = v;
        }
        __syncwarp(peers);
        if ((peers & lt) == 0u) cnt[r] = at + __popc(peers);
      }
      if (km && wpos >= 0) wpos += __popc(km);
      __syncwarp();
      const int rest = qn - take;
      const int mr = lane < rest ? (int)qrow[take + lane] : 0, mc = lane < rest ? qcol[take + lane] : 0;
      __syncwarp();
      if (lane < rest) { qrow[lane] = (unsigned char)mr; qcol[lane] = mc; }
      qn = rest;
      __syncwarp();
    };
    // run the first `take` pending look-ups, one per lane; the hits join the evaluation queue in look-up order
    int tn = 0;
    auto tflush = [&](int take) {
      const bool mine = lane < take;
      const int r = mine ? (int)tr[lane] : 0;
      const int g = mine ? tg[lane] : 0;
      const u64 b_row = __shfl_sync(full, br, r);
      int found = -1;
      if (mine) found = dh_find_beta(dets, __ldg(gstart + g), __ldg(gstart + g + 1), b_row);
      const unsigned m = __ballot_sync(full, found >= 0);
      if (m) {  // warp-uniform
        if (found >= 0) { const int idx = qn + __popc(m & lt); DH_CHECK(idx < 64); qrow[idx] = (unsigned char)r; qcol[idx] = found; }
        qn += __popc(m);
        __syncwarp();
        if (qn >= 32) flush(32);
      }
      const int rest = tn - take;
      const int mr = lane < rest ? (int)tr[take + lane] : 0, mg = lane < rest ? tg[take + lane] : 0;
      __syncwarp();
      if (lane < rest) { tr[lane] = (unsigned char)mr; tg[lane] = mg; }
      tn = rest;
      __syncwarp();
    };
    // runs of equal alpha among the 32 rows (S is sorted by alpha first)
    const u64 prev = __shfl_up_sync(full, ar, 1);
    const unsigned runs = __ballot_sync(full, have && (lane == 0 || ar != prev));
    const unsigned havem = __ballot_sync(full, have);
    for (int h0 = 0; h0 < ngroups; h0 += 32) {
      const int hq = h0 + lane;
      const u64 ah = hq < ngroups ? __ldg(galpha + hq) : 0ull;
      const int gs = hq < ngroups ? __ldg(gstart + hq) : 0, ge = hq < ngroups ? __ldg(gstart + hq + 1) : 0;
      for (unsigned rm = runs; rm;) {
        const int r0 = __ffs(rm) - 1;
        rm &= rm - 1;
        const int r1 = rm ? __ffs(rm) - 1 : 32 - __clz(havem);  // rows r0 .. r1-1 share one alpha string
        const u64 a_run = __shfl_sync(full, ar, r0);
        const int da = __popcll(a_run ^ ah);
        unsigned hm = __ballot_sync(full, hq < ngroups && da <= 4);
        if (!hm) continue;
        const unsigned hm4 = __ballot_sync(full, hq < ngroups && da == 4);
        if (hm == hm4) {
          // Every group of this chunk within reach is an alpha DOUBLE away (the common case: ~1500 such groups per run against ~50
          // an alpha single away): only the determinant with the row's own beta string connects, so that one string is looked
          // up in the group (sorted by beta) instead of the warp scanning the group.
          if (r1 - r0 >= 8) {
            // a long run: the lanes are its rows, one group at a time (ascending)
            for (unsigned gm = hm4; gm;) {
              const int hh = __ffs(gm) - 1;
              gm &= gm - 1;
              const int js = __shfl_sync(full, gs, hh), je = __shfl_sync(full, ge, hh);
              int found = -1;
              if (lane >= r0 && lane < r1) found = dh_find_beta(dets, js, je, br);
              const unsigned m = __ballot_sync(full, found >= 0);
              if (m) {  // warp-uniform
                if (found >= 0) { const int idx = qn + __popc(m & lt); DH_CHECK(idx < 64); qrow[idx] = (unsigned char)lane; qcol[idx] = found; }
                qn += __popc(m);
                __syncwarp();
                if (qn >= 32) flush(32);
              }
            }
          } else {
            // a short run: (row, group) look-ups are queued and run 32 at a time, whatever run and chunk they come from.  A row's
            // look-ups enter the queue in ascending group order and leave it in that order, so its columns stay ascending.
            const int k = __popc(hm4);
            for (int r = r0; r < r1; ++r) {
              if ((hm4 >> lane) & 1u) { const int idx = tn + __popc(hm4 & lt); DH_CHECK(idx < 64); tg[idx] = hq; tr[idx] = (unsigned char)r; }
              tn += k;
              __syncwarp();
              if (tn >= 32) tflush(32);
            }
          }
          continue;
        }
        while (tn > 0) tflush(tn < 32 ? tn : 32);  // the groups below are handled at once: what was found before them goes first
        while (hm) {  // groups within reach of this run, ascending
          const int hh = __ffs(hm) - 1;
          hm &= hm - 1;
          const int dmax = 4 - __shfl_sync(full, da, hh);
          const int js = __shfl_sync(full, gs, hh), je = __shfl_sync(full, ge, hh);
          const int M = je - js, R = r1 - r0;
          if (dmax == 0) {
            // an alpha double in a chunk that also holds closer groups: kept in group order; the lanes are the rows of the run
            int found = -1;
            if (lane >= r0 && lane < r1) found = dh_find_beta(dets, js, je, br);
            const unsigned m = __ballot_sync(full, found >= 0);
            if (m) {  // warp-uniform
              if (found >= 0) { const int idx = qn + __popc(m & lt); DH_CHECK(idx < 64); qrow[idx] = (unsigned char)lane; qcol[idx] = found; }
              qn += __popc(m);
              __syncwarp();
              if (qn >= 32) flush(32);
            }
          } else if (M <= 32 && R > 1) {
            // a small group against a run of several rows: the lanes cover the R x M cross product (row-major, so that a
            // row's columns still come in ascending order), instead of M of 32 lanes once per row
            const u64 bj = lane < M ? __ldg(dets + 2 * (int64_t)(js + lane) + 1) : 0ull;
            const unsigned inv = (65536u + (unsigned)M - 1u) / (unsigned)M;  // t / M == (t * inv) >> 16 for t < 1024, M <= 32
            const int T = R * M;
            for (int t0 = 0; t0 < T; t0 += 32) {
              const int t = t0 + lane;
              const int q = (int)(((unsigned)t * inv) >> 16), mm = t - q * M;
              const int r = r0 + (t < T ? q : 0);
              const u64 b_row = __shfl_sync(full, br, r);
              const u64 b_col = __shfl_sync(full, bj, t < T ? mm : 0);
              const bool hit = t < T && __popcll(b_row ^ b_col) <= dmax;
              const unsigned m = __ballot_sync(full, hit);
              if (m) {  // warp-uniform
                if (hit) { const int idx = qn + __popc(m & lt); DH_CHECK(idx < 64); qrow[idx] = (unsigned char)r; qcol[idx] = js + mm; }
                qn += __popc(m);
                __syncwarp();
                if (qn >= 32) flush(32);
              }
            }
          } else {
            for (int c0 = js; c0 < je; c0 += 32) {
              const int j = c0 + lane;
              const u64 bj = j < je ? __ldg(dets + 2 * (int64_t)j + 1) : 0ull;
              for (int r = r0; r < r1; ++r) {  // every row of the run against these 32 columns
                const u64 b_row = __shfl_sync(full, br, r);
                const bool hit = j < je && __popcll(b_row ^ bj) <= dmax;
                const unsigned m = __ballot_sync(full, hit);
                if (m) {  // warp-uniform
                  if (hit) { const int idx = qn + __popc(m & lt); DH_CHECK(idx < 64); qrow[idx] = (unsigned char)r; qcol[idx] = j; }
                  qn += __popc(m);
                  __syncwarp();
                  if (qn >= 32) flush(32);
                }
              }
            }
          }
        }
      }
    }
    while (tn > 0) tflush(tn < 32 ? tn : 32);
    if (qn > 0) flush(qn);
    if (have) row_cnt[row] = cnt[lane];
    __syncwarp();
  }
  if (lane == 0 && wpos >= 0 && wend > 0) bused[(wend - 1) / kArenaBlk] = (int)(wpos - (wend - kArenaBlk));
  for (int o = 16; o > 0; o >>= 1) evaluated += __shfl_xor_sync(full, evaluated, o);
  if (lane == 0 && evaluated) atomicAdd(counters + 1, evaluated);
}

// arena -> CSR: entry e of a block's used part goes to row_ptr[row] + place in the row
__global__ void pair_scatter_kernel(const u64* __restrict__ akey, const int* __restrict__ acol, const double* __restrict__ aval,
                                    const int* __restrict__ bused, int64_t n_arena, const int64_t* __restrict__ row_ptr,
                                    int* __restrict__ col, double* __restrict__ val) {
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n_arena; e += (int64_t)gridDim.x * blockDim.x) {
    if ((int)(e % kArenaBlk) >= bused[e / kArenaBlk]) continue;
    const u64 key = akey[e];
    const int64_t dst = row_ptr[key >> 32] + (int64_t)(key & 0xffffffffull);
    DH_CHECK(dst < row_ptr[(key >> 32) + 1]);
    col[dst] = acol[e]; val[dst] = aval[e];
  }
}

}  // namespace

// H_SS by excitation degree.  Same results as the list-walking build (dh_ham_build's other organisation): CSR owned by the
// context, columns ascending, diagonal always present.
dh_status dh_pair_build(detham_ctx* c, double eps) {
  const int64_t nd = c->nd;
  const HbLists* L = nullptr;
  dh_status st = dh_get_lists(c, 0, &L); if (st != DH_OK) return st;
  EnumParams P = dh_make_params(c, L);
  auto grow = [&](void** p, int64_t* cap, int64_t need, size_t elem) -> dh_status {
    if (*cap >= need) return DH_OK;
    if (*p) cudaFree(*p);
    *p = nullptr; *cap = 0;
    DH_CUDA(c, cudaMalloc(p, (size_t)need * elem));
    *cap = need;
    return DH_OK;
  };
  st = grow(reinterpret_cast<void**>(&c->row_cnt), &c->row_cnt_cap, nd, sizeof(int)); if (st != DH_OK) return st;
  if (c->row_cap < nd) {
    if (c->row_ptr) cudaFree(c->row_ptr);
    c->row_ptr = nullptr; c->row_cap = 0;
    DH_CUDA(c, cudaMalloc(&c->row_ptr, (nd + 1) * sizeof(int64_t)));
    c->row_cap = nd;
  }
  st = grow(reinterpret_cast<void**>(&c->pair_diag), &c->pair_diag_cap, nd, sizeof(double)); if (st != DH_OK) return st;
  c->nnz = -1;
  int64_t* h = reinterpret_cast<int64_t*>(c->pinned);
  const unsigned nb256 = (unsigned)((nd + 1 + 255) / 256);
  DH_TICK(c, 0);
  // ---- alpha groups of the sorted S
  group_flag_kernel<<<nb256, 256, 0, c->stream>>>(c->dets, nd, c->row_cnt);
  excl_scan_kernel<<<1, 1024, 0, c->stream>>>(c->row_cnt, nd, c->row_ptr);
  DH_CUDA(c, cudaGetLastError());
  DH_CUDA(c, cudaMemcpyAsync(h, c->row_ptr + nd, sizeof(int64_t), cudaMemcpyDeviceToHost, c->stream));
  DH_CUDA(c, cudaStreamSynchronize(c->stream));
  const int64_t ng = h[0];
  st = grow(reinterpret_cast<void**>(&c->pair_galpha), &c->pair_group_cap, ng + 1, sizeof(u64)); if (st != DH_OK) return st;
  if (c->pair_gstart_cap < ng + 1) {
    if (c->pair_gstart) cudaFree(c->pair_gstart);
    c->pair_gstart = nullptr; c->pair_gstart_cap = 0;
    DH_CUDA(c, cudaMalloc(&c->pair_gstart, (ng + 1) * sizeof(int)));
    c->pair_gstart_cap = ng + 1;
  }
  group_fill_kernel<<<nb256, 256, 0, c->stream>>>(c->dets, nd, c->row_cnt, c->row_ptr, c->pair_galpha, c->pair_gstart);
  pair_diag_kernel<<<(unsigned)((nd + 127) / 128), 128, 0, c->stream>>>(c->n, c->J, c->JK, c->hd, c->e_core, c->dets, nd, c->pair_diag);
  DH_CUDA(c, cudaGetLastError());
  // ---- one pass into the arena (sized from the previous build; a guess the first time), row scan, scatter
  const int64_t nblk = (nd + 31) / 32;
  int64_t want = (nblk + kPairWarps - 1) / kPairWarps;
  const int grid = (int)(want < (int64_t)c->sm_count * 8 ? want : (int64_t)c->sm_count * 8);
  const int64_t slack = (int64_t)grid * kPairWarps * kArenaBlk;  // every warp may leave one block partly used
  int* overflow = reinterpret_cast<int*>(c->dcount + 8);
  int64_t want_arena = c->arena_cap;
  if (want_arena <= 0) {  // first build of the context: room for 1024 entries per row if a quarter of the free memory allows it
    size_t free_b = 0, total_b = 0;
    DH_CUDA(c, cudaMemGetInfo(&free_b, &total_b));
    const int64_t by_mem = (int64_t)(free_b / 4 / 20);  // 20 bytes per arena entry (tag, column, value)
    want_arena = std::max<int64_t>(nd * 64 + slack, std::min<int64_t>(nd * 1024 + slack, by_mem));
  }
  int64_t nnz = 0, n_arena = 0;
  double ms_pass = 0.0;
  for (int attempt = 0;; ++attempt) {
    if (c->arena_cap < want_arena) {
      if (c->acol) cudaFree(c->acol);
      if (c->aval) cudaFree(c->aval);
      c->acol = nullptr; c->aval = nullptr; c->arena_cap = 0;
      DH_CUDA(c, cudaMalloc(&c->acol, want_arena * sizeof(int)));
      DH_CUDA(c, cudaMalloc(&c->aval, want_arena * sizeof(double)));
      c->arena_cap = want_arena;
    }
    st = grow(reinterpret_cast<void**>(&c->pair_akey), &c->pair_akey_cap, c->arena_cap, sizeof(u64)); if (st != DH_OK) return st;
    st = grow(reinterpret_cast<void**>(&c->pair_bused), &c->pair_bused_cap, c->arena_cap / kArenaBlk + 1, sizeof(int)); if (st != DH_OK) return st;
    DH_CUDA(c, cudaMemsetAsync(c->dcount, 0, 16 * sizeof(u64), c->stream));
    if (attempt > 0) DH_TICK(c, 0);
    pair_kernel<<<grid, kPairWarps * 32, 0, c->stream>>>(P, c->dets, nd, eps, c->pair_galpha, c->pair_gstart, (int)ng, c->pair_diag, c->row_cnt,
                                                        c->pair_akey, c->acol, c->aval, c->pair_bused, c->arena_cap, c->dcount, overflow);
    excl_scan_kernel<<<1, 1024, 0, c->stream>>>(c->row_cnt, nd, c->row_ptr);
    DH_CUDA(c, cudaGetLastError());
    DH_TICK(c, 1);
    DH_CUDA(c, cudaMemcpyAsync(h, c->row_ptr + nd, sizeof(int64_t), cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(c, cudaMemcpyAsync(h + 1, c->dcount, 3 * sizeof(u64), cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(c, cudaMemcpyAsync(h + 5, overflow, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(c, cudaStreamSynchronize(c->stream));
    ms_pass += dh_elapsed(c, 0, 1);
    nnz = h[0];
    n_arena = h[3];
    if (!*reinterpret_cast<int*>(h + 5)) break;
    if (attempt >= 1) return DH_ENOMEM;  // cannot happen: the second attempt is sized from the exact count
    want_arena = nnz + nnz / 32 + slack;  // a block is closed when the next batch of <= 32 entries does not fit
  }
  if (c->csr_cap < nnz) {
    if (c->col) cudaFree(c->col);
    if (c->val) cudaFree(c->val);
    c->col = nullptr; c->val = nullptr; c->csr_cap = 0;
    const int64_t cap = nnz > 0 ? nnz : 1;
    DH_CUDA(c, cudaMalloc(&c->col, cap * sizeof(int)));
    DH_CUDA(c, cudaMalloc(&c->val, cap * sizeof(double)));
    c->csr_cap = cap;
  }
  DH_TICK(c, 2);
  pair_scatter_kernel<<<c->sm_count * 16, 256, 0, c->stream>>>(c->pair_akey, c->acol, c->aval, c->pair_bused, n_arena, c->row_ptr, c->col, c->val);
  DH_CUDA(c, cudaGetLastError());
  DH_TICK(c, 3);
  DH_CUDA(c, cudaEventSynchronize(c->ev[3]));
  (void)ms_pass;
  c->ctr.ms_build_count = ms_pass;
  c->ctr.ms_build_fill = dh_elapsed(c, 2, 3);
  c->ctr.build_generated = h[2];  // elements evaluated (pairs of S within a double excitation of each other)
  c->ctr.nnz = nnz;
  c->ctr.build_pairs = 1;
  c->nnz = nnz;
  return DH_OK;
}
