// pt2 (a8, a9): external-determinant deduplication in an HBM open-addressing hash on 128-bit keys and the
// Epstein-Nesbet reduction (Eq. 13 second term; screening Eq. 14 / PAPER.md:219-227).
#include <math.h>
#include <stdio.h>
#include <stdlib.h>

#include <cmath>

#include "pt2_common.cuh"

EnumParams dh_make_params(detham_ctx* c, const HbLists* L);

namespace {

constexpr int kWarpsPerCta = 8;
constexpr int kFine = 1 << DH_MAX_PBITS;  // finest class histogram
// Tables beyond this size run region-binned passes (if the record pool fits).  Round 1 put the line at 32 GB (H2O-shaped, 15 GB:
// binned 17.5 ms against 12.8 ms direct); with this round's append it is lower: H2O-shaped 11.5 ms binned against 13.7 ms direct,
// N2-shaped sweep 1e4 (18.5 GB) 17.3 against 23.0 ms; H2O-shaped prefixes with 9.3 / 6.2 / 3.9 GB tables 7.0 / 5.0 / 3.4 ms against
// 8.5 / 6.2 / 4.5 ms.  The line stays at 8 GB, below every table of the BASELINE configurations that is not L2-sized.
constexpr int64_t kBinnedTableBytes = 8ll << 30;

// Slot (pt2_common.cuh): one 32-byte sector per external.  Members of S are pre-inserted with v = NaN.

__device__ __forceinline__ double member_flag() { return __longlong_as_double(0x7ff8000000000001ll); }


// ---------------------------------------------------------------- class histogram (pass planning)
// kExact = false: pass planning - singles are counted without being evaluated (an upper bound is all the planner needs).
// kExact = true: the exact number of screen-passing excitations (detham_count_screened): every single is evaluated.
template <bool kExact>
struct CountSink {
  static constexpr bool kLookupFirst = !kExact;
  static constexpr bool kLazySign = true;     // only counts
  unsigned* hist;
  __device__ __forceinline__ bool pre(u64, u64, u64 z) { atomicAdd(hist + ((unsigned)z & (kFine - 1)), 1u); return false; }
  __device__ __forceinline__ void emit(bool act, u64, u64, u64 z, double, int, int, int, int, int, int) {
    if (act) atomicAdd(hist + ((unsigned)z & (kFine - 1)), 1u);
  }
};

template <bool kExact>
__global__ void __launch_bounds__(kWarpsPerCta * 32)
count_kernel(EnumParams P, const u64* __restrict__ dets, const double* __restrict__ psi, int64_t nd, int64_t stride,
             double eps2, u64* counters, u64* __restrict__ hist) {
  extern __shared__ __align__(16) unsigned char smem[];
  CtaTables T = dh_cta_stage(P, smem);
  size_t off = (dh_cta_table_bytes(P.n) + 15) & ~(size_t)15;
  WarpScratch* wsp = reinterpret_cast<WarpScratch*>(smem + off);
  unsigned* sh = reinterpret_cast<unsigned*>(smem + off + kWarpsPerCta * sizeof(WarpScratch));
  for (int t = threadIdx.x; t < kFine; t += blockDim.x) sh[t] = 0;
  __syncthreads();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  WarpScratch& ws = wsp[warp];
  CountSink<kExact> sink{sh};
  for (;;) {
    u64 row = 0;
    if (lane == 0) row = atomicAdd(counters, 1ull);
    row = __shfl_sync(0xffffffffu, row, 0) * (u64)stride;  // every stride-th source (stride 1 = exact histogram)
    if ((int64_t)row >= nd) break;
    const double p = psi ? psi[row] : 1.0;  // no amplitudes: the amplitude-free screen of ham_build (tau = eps2)
    const u64 da = dets[2 * row], db = dets[2 * row + 1];
    u64 zsrc = 0;
    if (lane == 0) { zsrc = dh_zobrist(da, db, T.Z); if (!kExact) atomicAdd(sh + ((unsigned)zsrc & (kFine - 1)), 1u); }
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

// ---------------------------------------------------------------- sources ordered by key class
// The sub-list a source reads for an occupied pair (i, j) in pass p is that of class p ^ class(source) ^ z(i) ^ z(j): the 32 warps
// of a CTA, which take consecutive sources, share sub-lists (and so L1 lines) only if their sources are of one class.  perm =
// the sources sorted by class (counting sort; the order inside a class does not matter).
__global__ void class_count_kernel(const u64* __restrict__ dets, int64_t nd, unsigned pmask, unsigned* __restrict__ hist) {
  __shared__ u64 Z[128];
  for (int t = threadIdx.x; t < 128; t += blockDim.x) Z[t] = dh_zword(t);
  __syncthreads();
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nd) return;
  atomicAdd(hist + ((unsigned)dh_zobrist(dets[2 * t], dets[2 * t + 1], Z) & pmask), 1u);
}
__global__ void class_fill_kernel(const u64* __restrict__ dets, int64_t nd, unsigned pmask, unsigned* __restrict__ cursor, int* __restrict__ perm) {
  __shared__ u64 Z[128];
  for (int t = threadIdx.x; t < 128; t += blockDim.x) Z[t] = dh_zword(t);
  __syncthreads();
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nd) return;
  perm[atomicAdd(cursor + ((unsigned)dh_zobrist(dets[2 * t], dets[2 * t + 1], Z) & pmask), 1u)] = (int)t;
}

// ---------------------------------------------------------------- members of S of this pass's class
__global__ void member_insert_kernel(const u64* __restrict__ dets, int64_t nd, unsigned pmask, unsigned pass, Slot* table,
                                     u64 cap, int rshift, int* overflow) {
  __shared__ u64 Z[128];
  for (int t = threadIdx.x; t < 128; t += blockDim.x) Z[t] = dh_zword(t);
  __syncthreads();
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nd) return;
  u64 a = dets[2 * t], b = dets[2 * t + 1];
  u64 z = dh_zobrist(a, b, Z);
  if (((unsigned)z & pmask) != pass) return;
  u64 slot = dh_table_slot(z, a, b, cap, rshift);
  for (int probes = 0;; ++probes) {
    Slot* sp = table + slot;
    Key128 old = dh_cas128(sp, Key128{0ull, 0ull}, Key128{a, b});
    if (old.a == 0ull && old.b == 0ull) { sp->v = member_flag(); return; }
    if (++slot == cap) slot = 0;
    if (probes > kProbeLimit) { *overflow = 1; return; }
  }
}

// ---------------------------------------------------------------- accumulate
// One warp per source determinant, one CTA per SM.  Per (source, pass):
//   singles  - candidates of this pass's key class are compacted into a small queue and evaluated 32 at a time
//              (reading Q5: every single is evaluated exactly, in the order of reading Q7);
//   doubles  - phase A: every occupied pair (i,j) looks up its class sub-list and finds, by a galloping search on the
//              magnitude-sorted values, the prefix with |value| >= tau (the paper's early exit, taken as
//              a search instead of a walk); empty prefixes are dropped and the lengths prefix-summed;
//              phase B: the concatenation of all prefixes is walked 32*kU entries at a time, so every lane holds an
//              entry whatever the individual prefix lengths are, and each lane issues kU independent table probes
//              before it waits on any of them.
constexpr int kChunk = 128;     // occupied pairs per phase-A chunk
// kAccWarps warps per CTA and kU table probes in flight per lane are template parameters of the kernel

struct FlatScratch {
  u64 zij[kChunk];               // partition word of the source with (i,j) removed
  int pref[kChunk + 1];          // exclusive prefix of the kept lengths
  int beg[kChunk];               // first list entry of the kept prefix
  unsigned short meta[kChunk];   // fam << 12 | i << 6 | j
  unsigned short sq[64];         // singles queue: s << 12 | i << 6 | a
  unsigned dq[64];               // doubles queue: list entry | pair of the chunk << 25
};

struct ProbeCtx {
  Slot* table; u64 cap;
  const CtaTables* T; const WarpScratch* ws; int n;
  double e0;
  unsigned contrib; int max_probe;
  int* overflow;
};

// v_a += H_ai psi_i; in expand mode (row f2) the slot's second payload word holds max_i |H_ai psi_i| (Eq. 14's score)
// instead of H_aa: the bit patterns of non-negative doubles order like the values, so an unsigned RED.MAX does it.
template <bool kExpand>
__device__ __forceinline__ void slot_add(Slot* sp, double cv) {
  atomicAdd(&sp->v, cv);
  if (kExpand) atomicMax(reinterpret_cast<u64*>(&sp->haa), (u64)__double_as_longlong(fabs(cv)));
}

// Resolve up to U candidates per lane: all pending slots are loaded before any is examined, all needed CAS are issued
// before any result is used.  A slot is {key, v, H_aa}; members of S carry the NaN flag in v and absorb nothing.
template <int U, bool kExpand>
__device__ __forceinline__ void probe_batch(ProbeCtx& pc, const u64 (&ka)[U], const u64 (&kb)[U], const double (&cv)[U],
                                            u64 (&slot)[U], const double (&haa)[U], unsigned pend) {
  if (!pend) return;
  int probes = 0;
  for (;;) {
    u64 k0[U], k1[U], vb[U], hb[U];
#pragma unroll
    for (int u = 0; u < U; ++u)
      if ((pend >> u) & 1u) { DH_CHECK(slot[u] < pc.cap); dh_ld256(pc.table + slot[u], k0[u], k1[u], vb[u], hb[u]); }
    unsigned cas = 0;
#pragma unroll
    for (int u = 0; u < U; ++u)
      if ((pend >> u) & 1u) {
        if (k0[u] == ka[u] && k1[u] == kb[u]) {
          if (vb[u] != (u64)0x7ff8000000000001ull) { slot_add<kExpand>(pc.table + slot[u], cv[u]); ++pc.contrib; }
          pend &= ~(1u << u);
        } else if ((k0[u] | k1[u]) == 0ull || (k0[u] == 0ull) != (k1[u] == 0ull)) {
          // empty - or one word still zero: the 256-bit load is not single-copy atomic against another thread's 128-bit
          // claim, so a half-written key is possible in principle; the CAS below returns the whole key atomically either way
          cas |= 1u << u;
        } else if (++slot[u] == pc.cap) {
          slot[u] = 0;
        }
      }
    if (cas) {
#pragma unroll
      for (int u = 0; u < U; ++u)
        if ((cas >> u) & 1u) {
          Key128 old = dh_cas128(pc.table + slot[u], Key128{0ull, 0ull}, Key128{ka[u], kb[u]});
          k0[u] = old.a; k1[u] = old.b;
        }
#pragma unroll
      for (int u = 0; u < U; ++u)
        if ((cas >> u) & 1u) {
          if ((k0[u] | k1[u]) == 0ull) {  // claimed: this thread also records H_aa
            if (!kExpand) pc.table[slot[u]].haa = haa[u];
            slot_add<kExpand>(pc.table + slot[u], cv[u]); ++pc.contrib;
            pend &= ~(1u << u);
          } else if (k0[u] == ka[u] && k1[u] == kb[u]) {  // lost the race to the same key, or came here through the half-zero check
            const u64 vb2 = *reinterpret_cast<volatile u64*>(&pc.table[slot[u]].v);  // members were flagged before this kernel started
            if (vb2 != (u64)0x7ff8000000000001ull) { slot_add<kExpand>(pc.table + slot[u], cv[u]); ++pc.contrib; }
            pend &= ~(1u << u);
          } else if (++slot[u] == pc.cap) {
            slot[u] = 0;
          }
        }
    }
    if (!pend) break;
    if (++probes > kProbeLimit) { *pc.overflow = 1; break; }
  }
  pc.max_probe = max(pc.max_probe, probes);
}

// Binned mode (tables far beyond L2): instead of probing the table, a contribution is appended as a 32-byte record
// {key, H_ai psi_i, H_aa} to this CTA's private segment of the bin its slot falls in (bin = slot >> shift: a contiguous
// region of the table).  pt2_merge_kernel then walks the bins in order, so the probes of the whole GPU stay inside a window
// of the table that fits L2 (profiles/r1_microbench.md, block C: 36-41 G/s against 15 G/s for random probes).  The position
// in the segment comes from a shared-memory counter: no global atomic.  A record that does not fit its segment is probed
// directly, as in the unbinned kernel.
struct BinCtx { Slot* pool; unsigned* cnt; unsigned seg_cap; int shift; unsigned nbins; };

template <int U>
__device__ __forceinline__ unsigned bin_batch(ProbeCtx& pc, const BinCtx& bc, const u64 (&ka)[U], const u64 (&kb)[U],
                                              const double (&cv)[U], const u64 (&slot)[U], const double (&haa)[U], unsigned pend) {
#pragma unroll
  for (int u = 0; u < U; ++u)
    if ((pend >> u) & 1u) {
      const unsigned bin = (unsigned)(slot[u] >> bc.shift);
      DH_CHECK(bin < bc.nbins);
      const unsigned p = atomicAdd(&bc.cnt[bin], 1u);
      if (p < bc.seg_cap) {
        dh_st256(bc.pool + ((u64)bin * gridDim.x + blockIdx.x) * bc.seg_cap + p, ka[u], kb[u], (u64)__double_as_longlong(cv[u]),
                 (u64)__double_as_longlong(haa[u]));
        pend &= ~(1u << u);
      }
    }
  return pend;
}

// decode the triangular index t = y(y-1)/2 + x, x < y
__device__ __forceinline__ void tri_decode(int t, int& x, int& y) {
  y = (int)((1.0f + sqrtf(1.0f + 8.0f * (float)t)) * 0.5f);
  while (y * (y - 1) / 2 > t) --y;
  while ((y + 1) * y / 2 <= t) ++y;
  x = t - y * (y - 1) / 2;
}

template <int kAccWarps, int kU, bool kExpand, bool kBinned = false>
__global__ void __launch_bounds__(kAccWarps * 32, 1)
pt2_accumulate_kernel(EnumParams P, const u64* __restrict__ dets, const double* __restrict__ psi, int64_t nd, double eps2,
                      unsigned pass, Slot* table, u64 cap, u64* counters /* [0] next row [1] gen [2] contrib [3] max probe */,
                      int* overflow, Slot* pool, unsigned* used, unsigned seg_cap, int bin_shift, int nbins,
                      const int* __restrict__ perm /* order in which the sources are taken, or NULL */) {
  extern __shared__ __align__(16) unsigned char smem[];
  CtaTables T = dh_cta_stage<false>(P, smem);
  size_t off = (dh_cta_light_bytes(P.n) + 15) & ~(size_t)15;
  WarpScratch* wsp = reinterpret_cast<WarpScratch*>(smem + off);
  FlatScratch* fsp = reinterpret_cast<FlatScratch*>(smem + off + kAccWarps * sizeof(WarpScratch));
  unsigned* bcnt = reinterpret_cast<unsigned*>(fsp + kAccWarps);  // [nbins] records this CTA appended per bin (binned mode)
  if (kBinned) {
    for (int t = threadIdx.x; t < nbins; t += blockDim.x) bcnt[t] = 0;
    __syncthreads();
  }
  const BinCtx bc{pool, bcnt, seg_cap, bin_shift, (unsigned)nbins};
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const unsigned lt = (1u << lane) - 1u;
  WarpScratch& ws = wsp[warp];
  FlatScratch& fs = fsp[warp];
  const int n = P.n, na = P.na, nb = P.nb;
  const unsigned pmask = (1u << P.pbits) - 1u;
  const int NP = 1 << P.pbits;
  const int nAA = na * (na - 1) / 2, nBB = nb * (nb - 1) / 2, npairs = nAA + nBB + na * nb;
  const int nva = n - na, nvb = n - nb, tot_a = na * nva, tot_s = tot_a + nb * nvb;
  ProbeCtx pc{table, cap, &T, &ws, n, 0.0, 0u, 0, overflow};
  u64 gen_total = 0, contrib_total = 0;
  for (;;) {
    u64 row = 0;
    if (lane == 0) row = atomicAdd(counters, 1ull);
    row = __shfl_sync(0xffffffffu, row, 0);
    if ((int64_t)row >= nd) break;
    int ovf = 0;
    if (lane == 0) ovf = *reinterpret_cast<volatile int*>(overflow);
    if (__shfl_sync(0xffffffffu, ovf, 0)) break;  // warp-uniform by construction
    if (perm) { row = (u64)perm[row]; DH_CHECK((int64_t)row < nd); }
    const double p = psi[row];
    if (p == 0.0) continue;  // reading Q6: a source with zero amplitude generates nothing
    const double tau = eps2 == 0.0 ? 0.0 : __ddiv_rn(eps2, fabs(p));
    const u64 da = dets[2 * row], db = dets[2 * row + 1];
    dh_fill_occ(P, ws, da, db, lane);
    pc.e0 = dh_fill_U(P, T, ws, lane);
    pc.contrib = 0u;
    unsigned gen = 0u;
    u64 zsrc = 0;
    if (lane == 0) zsrc = dh_zobrist(da, db, T.Z);
    zsrc = __shfl_sync(0xffffffffu, zsrc, 0);

    // ---- singles
    {
      int qn = 0;
      for (int t0 = 0; t0 < tot_s + 32; t0 += 32) {
        const bool last = t0 >= tot_s;
        if (!last) {
          const int t = t0 + lane;
          bool in = t < tot_s;
          unsigned code = 0;
          if (in) {
            const int s = t >= tot_a ? 1 : 0, tt = s ? t - tot_a : t, nv = s ? nvb : nva;
            const int i = ws.occ[s][tt / nv], a = ws.vir[s][tt % nv];
            const u64 z = zsrc ^ T.Z[64 * s + i] ^ T.Z[64 * s + a];
            in = ((unsigned)z & pmask) == pass;
            code = ((unsigned)s << 12) | ((unsigned)i << 6) | (unsigned)a;
          }
          const unsigned m = __ballot_sync(0xffffffffu, in);
          DH_CHECK(qn + __popc(m) <= 64);
          if (in) fs.sq[qn + __popc(m & lt)] = (unsigned short)code;
          qn += __popc(m);
          __syncwarp();
        }
        if (qn >= 32 || (last && qn > 0)) {
          const int take = qn >= 32 ? 32 : qn;
          u64 ka[1] = {da}, kb[1] = {db}, slot[1] = {0};
          double cv[1] = {0.0};
          double haa[1] = {0.0};
          unsigned pend = 0u;
          if (lane < take) {
            const unsigned code = fs.sq[qn - take + lane];
            const int s = (int)(code >> 12), i = (int)((code >> 6) & 63u), a = (int)(code & 63u);
            const u64 w = s ? db : da;
            const double v = dh_single_value(P, ws, w, s, i, a);
            if (v != 0.0 && fabs(v) >= tau) {
              const u64 nw = (w ^ (1ull << i)) | (1ull << a);
              if (s == 0) ka[0] = nw; else kb[0] = nw;
              const u64 z = zsrc ^ T.Z[64 * s + i] ^ T.Z[64 * s + a];
              slot[0] = dh_table_slot(z, ka[0], kb[0], cap, bin_shift);
              cv[0] = v * p;
              if (!kExpand) haa[0] = dh_excited_diag(T, ws, n, pc.e0, 0, s, i, 0, a, 0);
              pend = 1u;
            }
          }
          __syncwarp();
          qn -= take;
          gen += pend;
          if (kBinned) pend = bin_batch<1>(pc, bc, ka, kb, cv, slot, haa, pend);
          probe_batch<1, kExpand>(pc, ka, kb, cv, slot, haa, pend);
        }
      }
    }

    // ---- doubles
    for (int qb = 0; qb < npairs; qb += kChunk) {
      const int qe = min(npairs, qb + kChunk);
      int cnt = 0, run = 0;
      // phase A: kept prefix of every pair's class sub-list
      for (int q0 = qb; q0 < qe; q0 += 32) {
        const int q = q0 + lane;
        int len = 0, beg = 0;
        unsigned pm = 0;
        u64 zij = 0;
        if (q < qe) {
          int fam, i, j, seg;
          if (q < nAA) { int x, y; tri_decode(q, x, y); fam = 0; i = ws.occ[0][x]; j = ws.occ[0][y]; seg = j * (j - 1) / 2 + i; zij = zsrc ^ T.Z[i] ^ T.Z[j]; }
          else if (q < nAA + nBB) { int x, y; tri_decode(q - nAA, x, y); fam = 1; i = ws.occ[1][x]; j = ws.occ[1][y]; seg = P.nss + j * (j - 1) / 2 + i; zij = zsrc ^ T.Z[64 + i] ^ T.Z[64 + j]; }
          else { const int r = q - nAA - nBB; fam = 2; i = ws.occ[0][r / nb]; j = ws.occ[1][r % nb]; seg = 2 * P.nss + i * n + j; zij = zsrc ^ T.Z[i] ^ T.Z[64 + j]; }
          const unsigned cls = ((unsigned)zij ^ pass) & pmask;
          const int64_t so = (int64_t)seg * NP + cls;
          beg = __ldg(P.sub_off + so);
          const int end = __ldg(P.sub_off + so + 1);
          int lo = beg, hi = end;
          if (tau != 0.0) {  // first index whose |value| < tau: gallop from the head (most kept prefixes are short), then bisect
            int pos = beg, step = 1;
            while (pos < end && fabs(__ldg(P.lval + pos)) >= tau) { lo = pos + 1; pos += step; step <<= 1; }
            hi = min(pos, end);
            while (lo < hi) {
              const int mid = (lo + hi) >> 1;
              if (fabs(__ldg(P.lval + mid)) >= tau) lo = mid + 1; else hi = mid;
            }
          } else {  // tau = 0: everything but exact zeros (reading Q8), which the |value|-descending order puts at the tail
            while (lo < hi) {
              const int mid = (lo + hi) >> 1;
              if (__ldg(P.lval + mid) != 0.0) lo = mid + 1; else hi = mid;
            }
          }
          len = lo - beg;
          pm = ((unsigned)fam << 12) | ((unsigned)i << 6) | (unsigned)j;
        }
        const unsigned m = __ballot_sync(0xffffffffu, len > 0);
        int x = len;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
        const int tot = __shfl_sync(0xffffffffu, x, 31);
        if (len > 0) {
          const int idx = cnt + __popc(m & lt);
          fs.pref[idx] = run + x - len; fs.beg[idx] = beg; fs.meta[idx] = (unsigned short)pm; fs.zij[idx] = zij;
        }
        cnt += __popc(m);
        run += tot;
      }
      if (lane == 0) fs.pref[cnt] = run;
      __syncwarp();
      // phase B: walk the concatenated prefixes 32 entries at a time.  Entries whose a or b is occupied in the source (about
      // 40 % on the Cr2-shaped config) are dropped first - one 2-byte load and a bit test - and the survivors queued, so that
      // value, phase, key, slot and H_aa are worked out, and the table probed, with every lane busy.
      const int TT = run;
      int qcur = 0, dqn = 0;
      for (int t0 = 0; t0 < TT + 32; t0 += 32) {
        const bool last = t0 >= TT;
        if (!last) {
          const int pe = (qcur + lane < cnt) ? fs.pref[qcur + lane + 1] - t0 : 0x7fffffff;  // end of pair qcur+lane, relative
          const unsigned bm = __reduce_or_sync(0xffffffffu, pe < 32 ? (1u << pe) : 0u);
          const int adv = __popc(__ballot_sync(0xffffffffu, pe <= 32));
          const int myq = qcur + __popc(bm & ((2u << lane) - 1u));
          qcur += adv;
          const int t = t0 + lane;
          bool act = false;
          unsigned ent = 0u;
          if (t < TT) {
            const int k = fs.beg[myq] + (t - fs.pref[myq]);
            const unsigned ab = __ldg(P.lab + k);
            const int a = (int)(ab & 0xFFu), b = (int)(ab >> 8);
            const unsigned fam = fs.meta[myq] >> 12;
            const u64 wa = fam == 1u ? db : da, wb = fam != 0u ? db : da;  // spin string of (i, a) and of (j, b)
            act = !(((wa >> a) | (wb >> b)) & 1ull);
            ent = (unsigned)k | ((unsigned)myq << 25);
          }
          const unsigned m = __ballot_sync(0xffffffffu, act);
          DH_CHECK(dqn + __popc(m) <= 64);
          if (act) fs.dq[dqn + __popc(m & lt)] = ent;
          dqn += __popc(m);
          __syncwarp();
        }
        if (dqn >= 32 || (last && dqn > 0)) {
          const int take = dqn >= 32 ? 32 : dqn;
          u64 ka[1] = {da}, kb[1] = {db}, slot[1] = {0};
          double cv[1] = {0.0};
          double haa[1] = {0.0};
          unsigned pend = 0u;
          if (lane < take) {
            const unsigned ent = fs.dq[dqn - take + lane];
            const int k = (int)(ent & 0x1FFFFFFu), myq = (int)(ent >> 25);
            const unsigned pm = fs.meta[myq];
            double v = __ldg(P.lval + k);
            const unsigned ab = __ldg(P.lab + k);
            const int a = (int)(ab & 0xFFu), b = (int)(ab >> 8);
            const int fam = (int)(pm >> 12), i = (int)((pm >> 6) & 63u), j = (int)(pm & 63u);
            const u64 zij = fs.zij[myq];
            if (fam < 2) {
              const u64 w = fam ? db : da;
              const u64 nw = (w ^ (1ull << i) ^ (1ull << j)) | (1ull << a) | (1ull << b);
              if (fam == 0) ka[0] = nw; else kb[0] = nw;
              const u64 z = zij ^ T.Z[64 * fam + a] ^ T.Z[64 * fam + b];
              // a+_a a+_b a_j a_i = (a+_b a_j)(a+_a a_i): phase(i->a on w) * phase(j->b on w with i->a applied)
              const int par = dh_parity_between(w, i, a) ^ dh_parity_between((w ^ (1ull << i)) | (1ull << a), j, b);
              if (par) v = -v;
              slot[0] = dh_table_slot(z, ka[0], kb[0], cap, bin_shift);
            } else {
              ka[0] = (da ^ (1ull << i)) | (1ull << a);
              kb[0] = (db ^ (1ull << j)) | (1ull << b);
              const u64 z = zij ^ T.Z[a] ^ T.Z[64 + b];
              if (dh_parity_between(da, i, a) ^ dh_parity_between(db, j, b)) v = -v;
              slot[0] = dh_table_slot(z, ka[0], kb[0], cap, bin_shift);
            }
            cv[0] = v * p;
            if (!kExpand) {  // O(1) diagonal update: the source's U vectors plus the entry's source-independent part (lists.cu)
              const int si = fam == 1, sj = fam != 0;
              haa[0] = pc.e0 - ws.U[si][i] - ws.U[sj][j] + ws.U[si][a] + ws.U[sj][b] + __ldg(P.lstat + k);
            }
            pend = 1u;
          }
          __syncwarp();
          dqn -= take;
          gen += pend;
          if (kBinned) pend = bin_batch<1>(pc, bc, ka, kb, cv, slot, haa, pend);
          probe_batch<1, kExpand>(pc, ka, kb, cv, slot, haa, pend);
        }
      }
      __syncwarp();
    }
    gen_total += gen;
    contrib_total += pc.contrib;
  }
  u64 g = gen_total, ct = contrib_total;
  int mp = pc.max_probe;
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
  if (kBinned) {
    __syncthreads();
    for (int t = threadIdx.x; t < nbins; t += blockDim.x) used[(size_t)t * gridDim.x + blockIdx.x] = min(bcnt[t], seg_cap);
  }
}

// Binned mode, second half: the records of bin b (one segment per accumulate CTA) are merged into the table region the bin
// covers.  The CTAs take (bin, segment) chunks from one global cursor in bin-major order, so at any time all probes of the
// GPU fall into one or two neighbouring regions (32 MB each at the default 2048 regions of a 60 GB table).  The probe itself is the
// unbinned kernel's; H_aa comes with the record.
__global__ void __launch_bounds__(1024, 2)
pt2_table_merge_kernel(const Slot* __restrict__ pool, const unsigned* __restrict__ used, unsigned seg_cap, int nbins, int nseg,
                 Slot* table, u64 cap, u64* counters /* [2] contrib [3] max probe [5] chunk cursor */, int* overflow, int rshift) {
  // work unit = kUnit consecutive records of one (bin, segment), taken per WARP from the global cursor in bin-major order: no
  // CTA barrier in the loop, and the ~9500 resident warps span three or four bins (128-record units were slower than the
  // CTA-wide chunks: 1e7 atomics per pass on the one cursor cost 18 ms)
  const int lane = threadIdx.x & 31;
  constexpr unsigned kUnit = 512;
  const unsigned nsub = (seg_cap + kUnit - 1u) / kUnit;
  const u64 nunits = (u64)nbins * nseg * nsub;
  unsigned contrib = 0; int max_probe = 0;
  for (;;) {
    u64 u = 0;
    if (lane == 0) u = atomicAdd(counters + 5, 1ull);
    u = __shfl_sync(0xffffffffu, u, 0);
    if (u >= nunits) break;
    const u64 q = u / nsub;                                       // segment (q % nseg) of bin (q / nseg)
    const unsigned lo = (unsigned)(u % nsub) * kUnit, n = used[q];
    if (lo >= n) continue;
    const unsigned hi = min(n, lo + kUnit);
    const Slot* src = pool + q * seg_cap;
    const u64 region = (q / nseg) << rshift;
    // Every lane works through its own records (lane, lane + 32, ...) at its own pace: one probe step per iteration for every
    // lane that has a record, the next record fetched as soon as the current one is placed.  (A loop over records with the probe
    // loop inside it leaves a warp waiting for its slowest lane at every record: 12.5 of 32 lanes active, measured.)
    unsigned t = lo + lane;
    bool have = false;
    u64 ka = 0, kb = 0, hh = 0, slot = 0;
    double cv = 0.0;
    int probes = 0;
    for (;;) {
      if (!have && t < hi) {
        u64 vv;
        dh_ld256_cs(src + t, ka, kb, vv, hh);
        // the record's region is the bin it was appended to; inside it the key's own hash gives the home slot (dh_table_slot)
        slot = region | (u64)(dh_key_hash(ka, kb) >> (32 - rshift));
        cv = __longlong_as_double((long long)vv);
        probes = 0;
        have = true;
        t += 32;
      }
      if (!__any_sync(0xffffffffu, have)) break;
      if (have) {
        u64 k0, k1, vb, hb;
        DH_CHECK(slot < cap);
        dh_ld256(table + slot, k0, k1, vb, hb);
        bool done = false;
        if (k0 == ka && k1 == kb) {
          if (vb != (u64)0x7ff8000000000001ull) { atomicAdd(&table[slot].v, cv); ++contrib; }
          done = true;
        } else if (k0 == 0ull || k1 == 0ull || k0 == ka || k1 == kb) {
          // empty - or a key seen half written (the 256-bit load is not ordered against another thread's 128-bit CAS): the CAS
          // both claims an empty slot and returns the key that is really there
          const Key128 old = dh_cas128(table + slot, Key128{0ull, 0ull}, Key128{ka, kb});
          if ((old.a | old.b) == 0ull) { table[slot].haa = __longlong_as_double((long long)hh); atomicAdd(&table[slot].v, cv); ++contrib; done = true; }
          else if (old.a == ka && old.b == kb) {
            // claimed by another thread in the meantime; a member of S is told apart by its flag, written right after its claim
            // by member_insert_kernel, which has finished before this kernel starts
            if (__double_as_longlong(*reinterpret_cast<volatile double*>(&table[slot].v)) != (long long)0x7ff8000000000001ull) { atomicAdd(&table[slot].v, cv); ++contrib; }
            done = true;
          }
        }
        if (!done) {
          if (++slot == cap) slot = 0;
          if (++probes > kProbeLimit) { *overflow = 1; done = true; }
        }
        if (done) { max_probe = max(max_probe, probes); have = false; }
      }
    }
  }
  u64 ct = contrib;
  for (int o = 16; o > 0; o >>= 1) { ct += __shfl_xor_sync(0xffffffffu, ct, o); max_probe = max(max_probe, __shfl_xor_sync(0xffffffffu, max_probe, o)); }
  if ((threadIdx.x & 31) == 0) { if (ct) atomicAdd(counters + 2, ct); atomicMax(counters + 3, (u64)max_probe); }
}

// ---------------------------------------------------------------- reduce: sum_a v_a^2 / (E_S - H_aa), and clear the table
__global__ void __launch_bounds__(256)
pt2_scan_kernel(Slot* table, u64 cap, double e_s, int n, const double* __restrict__ J, const double* __restrict__ JK,
                const double* __restrict__ hd, double e_core, double small_den, double* __restrict__ part /* [grid][4]: sum, sum_abs, min_den, count */) {
  double sum = 0.0, sabs = 0.0, mden = INFINITY, cnt = 0.0;
  constexpr int V = 4;  // independent 32-byte loads in flight per thread
  const u64 stride = (u64)gridDim.x * blockDim.x;
  for (u64 t0 = (u64)blockIdx.x * blockDim.x + threadIdx.x; t0 < cap; t0 += V * stride) {
    u64 x[V], y[V], z[V], w[V];
#pragma unroll
    for (int k = 0; k < V; ++k) {
      x[k] = y[k] = z[k] = w[k] = 0ull;
      const u64 t = t0 + k * stride;
      if (t < cap) dh_ld256_cs(table + t, x[k], y[k], z[k], w[k]);
    }
#pragma unroll
    for (int k = 0; k < V; ++k) {
      if (x[k] | y[k]) {
        if (z[k] != (u64)0x7ff8000000000001ull) {
          double v = __longlong_as_double((long long)z[k]), den = e_s - __longlong_as_double((long long)w[k]);
          // The slot's H_aa came from the O(1) update of whichever source claimed it first, so it carries that source's
          // rounding (~1e-13).  Where the denominator is small enough to amplify that, take H_aa from the key alone:
          // the same value in every run and for every partitioning (a few externals in a million).
          if (fabs(den) < small_den) den = e_s - dh_diag_from_scratch(n, J, JK, hd, e_core, x[k], y[k]);
          double term = v * v / den;
          sum += term; sabs += fabs(term); mden = fmin(mden, fabs(den)); cnt += 1.0;
        }
        dh_st256_zero(table + t0 + k * stride);
      }
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

// expand mode (row f2): move every external of this pass {key, v_a, score_a} to the output arrays (order arbitrary: the
// caller sorts by key afterwards) and clear the table.  Warp-aggregated: one atomic per warp and step.
__global__ void __launch_bounds__(256)
pt2_compact_kernel(Slot* table, u64 cap, u64* __restrict__ keys_out, double* __restrict__ v_out, double* __restrict__ score_out,
                   u64 out_cap, u64* cursor) {
  const u64 stride = (u64)gridDim.x * blockDim.x;
  const int lane = threadIdx.x & 31;
  const u64 cap_pad = (cap + 31) & ~(u64)31;
  for (u64 t = (u64)blockIdx.x * blockDim.x + threadIdx.x; t < cap_pad; t += stride) {
    u64 x = 0, y = 0, z = 0, w = 0;
    if (t < cap) dh_ld256_cs(table + t, x, y, z, w);
    const bool occ = (x | y) != 0ull;
    const bool ext = occ && z != (u64)0x7ff8000000000001ull;
    const unsigned m = __ballot_sync(0xffffffffu, ext);
    u64 base = 0;
    if (lane == 0 && m) base = atomicAdd(cursor, (u64)__popc(m));
    base = __shfl_sync(0xffffffffu, base, 0);
    if (ext) {
      const u64 pos = base + __popc(m & ((1u << lane) - 1u));
      if (pos < out_cap) {
        keys_out[2 * pos] = x; keys_out[2 * pos + 1] = y;
        if (v_out) v_out[pos] = __longlong_as_double((long long)z);
        if (score_out) score_out[pos] = __longlong_as_double((long long)w);
      }
    }
    if (occ) dh_st256_zero(table + t);
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
  static constexpr bool kLazySign = false;
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
  out[t] = dh_diag_from_scratch(n, J, JK, hd, e_core, dets[2 * t], dets[2 * t + 1]);
}

}  // namespace

static dh_status ensure_table(detham_ctx* c, int64_t slots) {
  if (c->table && c->table_slots >= slots) return DH_OK;
  if (c->table) cudaFree(c->table);
  c->table = nullptr; c->table_slots = 0;
  DH_CUDA(c, cudaMalloc(&c->table, (size_t)slots * sizeof(Slot)));
  DH_CUDA(c, cudaMemsetAsync(c->table, 0, (size_t)slots * sizeof(Slot), c->stream));  // the scan keeps it zero afterwards
  c->table_slots = slots;
  return DH_OK;
}

// One attempt at the whole PT2 with 2^pbits key partitions and a table of `slots` slots.  `adapt`: after pass 0 the
// capacity used by the later passes is shrunk to (distinct keys of pass 0) / load, which cuts the scan traffic when the
// table was sized from the contribution count (an upper bound of the distinct keys).
// `pilot` (may be NULL): run pass 0 only and return {distinct externals, milliseconds} - the planner's probe of how many
// contributions share an external.
struct ExpandOut { u64* keys; double* v; double* score; u64 cap; u64* cursor; };  // device buffers of expand mode

// `est_pass` (0 = unknown): upper estimate of the contributions of one pass; with it, and a table far beyond L2, the passes run
// binned: the accumulate kernel appends records to per-region segments (bin_batch), pt2_table_merge_kernel probes them region
// by region.
static dh_status pt2_attempt(detham_ctx* c, const double* psi, double e_s, double eps2, int pbits, int64_t slots, bool adapt,
                             double load, double* out, double* pilot = nullptr, const ExpandOut* ex = nullptr, double est_pass = 0.0,
                             bool force_binned = false) {
  const int64_t nd = c->nd;
  dh_status st = ensure_table(c, slots); if (st != DH_OK) return st;
  Slot* table = reinterpret_cast<Slot*>(c->table);
  const HbLists* L = nullptr;
  st = dh_get_lists(c, pbits, &L); if (st != DH_OK) return st;
  EnumParams P = dh_make_params(c, L);
  // launch shape: 32 warps per CTA, one probe in flight per lane.  Measured on B200 (round 1): more warps per SM help
  // (Cr2-shaped accumulate 1419 / 1084 / 1025 / 994 ms at 16 / 24 / 28 / 32 warps), more probes in flight per lane do not.
  const int warps = 32;
  int64_t want = (nd + warps - 1) / warps;
  const int grid = (int)(want < (int64_t)c->sm_count ? want : (int64_t)c->sm_count);
  // binned passes: table beyond kBinnedTableBytes, an estimate to size the record pool with, every SM busy, not expand / probe
  // (measured, round 1: H2O-shaped, 15 GB table, 5 contributions per external: 17.5 ms binned against 12.8 ms direct; N2-shaped,
  // 60 GB: 143 against 152 ms; Cr2-shaped: 5.9 against 7.4 s).  opt.table_regions: -1 never, > 0 always, with that many regions
  // at most (the region size is a power of two of slots; 2048 was the best of a sweep on Cr2-shaped).
  const int max_bins = c->opt.table_regions > 0 ? c->opt.table_regions : 2048;
  bool binned = !ex && !pilot && est_pass > 0.0 && grid == c->sm_count && c->opt.table_regions >= 0 &&
                (c->opt.table_regions > 0 || force_binned || slots * (int64_t)sizeof(Slot) > kBinnedTableBytes);
  unsigned* pool_used = nullptr;
  if (binned) {
    // the pool holds the records of one pass: 20 % head room over the estimate (an upper bound already) plus 64 records per
    // segment; it is divided evenly over the pass's (bin, CTA) segments, and what does not fit a segment is probed directly
    const double pool_frac = c->opt.stream_pool_frac > 0.0 ? c->opt.stream_pool_frac : 1.2;
    const int64_t bytes = (int64_t)((est_pass * pool_frac + 64.0 * max_bins * grid) * sizeof(Slot));
    size_t free_b = 0, total_b = 0;
    DH_CUDA(c, cudaMemGetInfo(&free_b, &total_b));
    if (c->pool_bytes < bytes) {
      if ((double)bytes > 0.95 * ((double)free_b + (double)c->pool_bytes)) binned = false;
      else {
        if (c->pool) cudaFree(c->pool);
        c->pool = nullptr; c->pool_bytes = 0;
        if (cudaMalloc(&c->pool, (size_t)bytes) != cudaSuccess) { cudaGetLastError(); binned = false; }
        else c->pool_bytes = bytes;
      }
    }
    const size_t ub = (size_t)max_bins * grid * sizeof(unsigned);
    if (binned && c->sflags_bytes < ub) {
      if (c->sflags) cudaFree(c->sflags);
      c->sflags = nullptr; c->sflags_bytes = 0;
      DH_CUDA(c, cudaMalloc(&c->sflags, ub));
      c->sflags_bytes = ub;
    }
    pool_used = reinterpret_cast<unsigned*>(c->sflags);
  }
  // sources in class order (see class_count_kernel); not for a single pass, where every source reads the same lists
  const int* perm = nullptr;
  if (pbits >= 1 && nd >= 4096 && nd < (1ll << 31)) {
    const int np = 1 << pbits;
    if (c->perm_cap < nd) {
      if (c->perm) cudaFree(c->perm);
      c->perm = nullptr; c->perm_cap = 0;
      DH_CUDA(c, cudaMalloc(&c->perm, nd * sizeof(int)));
      c->perm_cap = nd;
    }
    unsigned* chist = reinterpret_cast<unsigned*>(c->hist);  // [kFine] u64 = room for 2 * kFine counters
    std::vector<unsigned> hh(np);
    DH_CUDA(c, cudaMemsetAsync(chist, 0, np * sizeof(unsigned), c->stream));
    class_count_kernel<<<(unsigned)((nd + 255) / 256), 256, 0, c->stream>>>(c->dets, nd, (unsigned)(np - 1), chist);
    DH_CUDA(c, cudaGetLastError());
    DH_CUDA(c, cudaMemcpyAsync(hh.data(), chist, np * sizeof(unsigned), cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(c, cudaStreamSynchronize(c->stream));
    unsigned run = 0;
    for (int k = 0; k < np; ++k) { const unsigned t = hh[k]; hh[k] = run; run += t; }
    DH_CUDA(c, cudaMemcpyAsync(chist, hh.data(), np * sizeof(unsigned), cudaMemcpyHostToDevice, c->stream));
    class_fill_kernel<<<(unsigned)((nd + 255) / 256), 256, 0, c->stream>>>(c->dets, nd, (unsigned)(np - 1), chist, c->perm);
    DH_CUDA(c, cudaGetLastError());
    DH_CUDA(c, cudaStreamSynchronize(c->stream));  // hh is a host temporary
    perm = c->perm;
  }
  auto acc_kernel = ex ? pt2_accumulate_kernel<32, 1, true> : (binned ? pt2_accumulate_kernel<32, 1, false, true> : pt2_accumulate_kernel<32, 1, false>);
  const size_t smem = ((dh_cta_light_bytes(c->n) + 15) & ~(size_t)15) + warps * (sizeof(WarpScratch) + sizeof(FlatScratch)) +
                      (binned ? max_bins * sizeof(unsigned) : 0);
  DH_CUDA(c, cudaFuncSetAttribute(acc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const double small_den = c->opt.small_den == 0.0 ? 1e-3 : (c->opt.small_den < 0.0 ? 0.0 : c->opt.small_den);

  const int nparts = 1 << pbits;
  const int sgrid_max = c->sm_count * 16;
  st = dh_ensure_red(c, 4 * ((int64_t)sgrid_max + 64) + 4 * (int64_t)(nparts + 1)); if (st != DH_OK) return st;
  double* results = c->red;                        // [nparts + 1][4]; row nparts = psi^T psi
  double* part = c->red + 4 * (int64_t)(nparts + 1);
  int* overflow = reinterpret_cast<int*>(c->dcount + 8);
  u64* hp = reinterpret_cast<u64*>(c->pinned);
  DH_CUDA(c, cudaMemsetAsync(c->dcount, 0, 32 * sizeof(u64), c->stream));

  norm2_kernel<<<64, 256, 0, c->stream>>>(psi, nd, part);
  final_reduce4_kernel<<<1, 256, 0, c->stream>>>(part, 64, results + 4 * nparts);
  DH_CUDA(c, cudaGetLastError());

  u64 gen = 0, contrib = 0, max_probe = 0;
  double ms_accum = 0.0, ms_scan = 0.0;
  int64_t cap = slots;
  for (int pass = 0; pass < nparts; ++pass) {
    const int64_t sblocks = (cap + 1023) / 1024;
    const int sgrid = (int)(sblocks < sgrid_max ? sblocks : sgrid_max);
    DH_CUDA(c, cudaMemsetAsync(c->dcount, 0, 8 * sizeof(u64), c->stream));
    DH_TICK(c, 2);
    int bin_shift = 0, nbins = 1;
    unsigned seg_cap = 0;
    int64_t pcap = cap;  // capacity this pass probes
    if (binned) {  // bins = contiguous table regions of 2^shift slots, at most max_bins of them; whole regions only
      // the regions cover `cap` rounded UP to whole regions where the allocation allows it (rounding down would raise the load)
      bin_shift = 10;
      while (((cap + (1ll << bin_shift) - 1) >> bin_shift) > max_bins) ++bin_shift;
      nbins = (int)((cap + (1ll << bin_shift) - 1) >> bin_shift);
      if (((int64_t)nbins << bin_shift) > slots) nbins = (int)(slots >> bin_shift);
      if (nbins < 1) { nbins = 1; bin_shift = 0; while ((2ll << bin_shift) <= slots) ++bin_shift; }
      pcap = (int64_t)nbins << bin_shift;
      seg_cap = (unsigned)(c->pool_bytes / ((int64_t)nbins * grid * (int64_t)sizeof(Slot)));
    }
    member_insert_kernel<<<(unsigned)((nd + 255) / 256), 256, 0, c->stream>>>(c->dets, nd, (unsigned)(nparts - 1), (unsigned)pass, table, (u64)pcap, bin_shift, overflow);
    acc_kernel<<<grid, warps * 32, smem, c->stream>>>(P, c->dets, psi, nd, eps2, (unsigned)pass, table, (u64)pcap, c->dcount, overflow,
                                                      reinterpret_cast<Slot*>(c->pool), pool_used, seg_cap, bin_shift, nbins, perm);
    if (binned) {
      DH_CUDA(c, cudaGetLastError());
      if (c->debug) DH_TICK(c, 5);
      pt2_table_merge_kernel<<<c->sm_count * 2, 1024, 0, c->stream>>>(reinterpret_cast<const Slot*>(c->pool), pool_used, seg_cap, nbins, grid, table,
                                                                     (u64)pcap, c->dcount, overflow, bin_shift);
    }
    DH_TICK(c, 3);
    if (ex && !pilot) {
      pt2_compact_kernel<<<sgrid, 256, 0, c->stream>>>(table, (u64)cap, ex->keys, ex->v, ex->score, ex->cap, ex->cursor);
      DH_CUDA(c, cudaMemsetAsync(results + 4 * pass, 0, 4 * sizeof(double), c->stream));
    } else {
      // binned passes may probe up to a whole region beyond `cap`: the scan covers what was probed
      pt2_scan_kernel<<<sgrid, 256, 0, c->stream>>>(table, (u64)(pcap > cap ? pcap : cap), e_s, c->n, c->J, c->JK, c->hd, c->e_core, small_den, part);
      final_reduce4_kernel<<<1, 256, 0, c->stream>>>(part, sgrid, results + 4 * pass);
    }
    DH_CUDA(c, cudaGetLastError());
    DH_TICK(c, 4);
    DH_CUDA(c, cudaMemcpyAsync(hp, c->dcount, 4 * sizeof(u64), cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(c, cudaMemcpyAsync(hp + 4, overflow, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(c, cudaMemcpyAsync(hp + 8, results + 4 * pass, 4 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(c, cudaStreamSynchronize(c->stream));
    ms_accum += dh_elapsed(c, 2, 3); ms_scan += dh_elapsed(c, 3, 4);
    if (c->debug && binned && pass == 3) fprintf(stderr, "[detham] pt2 pass 3: append %.1f ms, merge %.1f ms, scan %.1f ms, %d regions of 2^%d slots\n", dh_elapsed(c, 2, 5), dh_elapsed(c, 5, 3), dh_elapsed(c, 3, 4), nbins, bin_shift);
    gen += hp[1]; contrib += hp[2]; if (hp[3] > max_probe) max_probe = hp[3];
    if (*reinterpret_cast<int*>(hp + 4)) return DH_ETABLEFULL;  // the scan above already cleared the table
    if (pilot) { pilot[0] = reinterpret_cast<double*>(hp + 8)[3]; pilot[1] = ms_accum + ms_scan; return DH_OK; }
    if (adapt && pass == 0 && nparts > 1) {
      const double u0 = reinterpret_cast<double*>(hp + 8)[3] + (double)nd / nparts;  // distinct externals + members of one class
      // binned passes probe in L2, where a load of 0.6 costs nothing (see the planner's note in pt2_run)
      const double need = (u0 + 8.0 * sqrt(u0) + 1024.0) / ((binned && c->opt.table_load <= 0.0 && u0 > 1e7) ? 0.6 : load);
      if (need < (double)cap) cap = (int64_t)need;
    }
  }
  std::vector<double> res(4 * (size_t)(nparts + 1));
  DH_CUDA(c, cudaMemcpyAsync(res.data(), results, res.size() * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  DH_CUDA(c, cudaStreamSynchronize(c->stream));
  const double norm2 = res[4 * (size_t)nparts];
  if (!(norm2 > 0.0) || !std::isfinite(norm2)) return DH_EINVAL;  // psi identically zero (or not finite): Eq. 13 has no value
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
  c->ctr.pt2_binned = binned ? 1 : 0;
  c->ctr.pt2_stream_bins = 0;
  c->ctr.pt2_sum_abs = sabs / norm2;
  c->ctr.pt2_min_abs_den = mden;
  c->ctr.ms_pt2_accum = ms_accum;
  c->ctr.ms_pt2_scan = ms_scan;
  return DH_OK;
}

void dh_launch_final_reduce4(const double* part, int nblk, double* out, cudaStream_t stream) {
  final_reduce4_kernel<<<1, 256, 0, stream>>>(part, nblk, out);
}

static dh_status pt2_run(detham_ctx* c, const double* psi, double e_s, double eps2, double* out, const ExpandOut* ex) {
  const int64_t nd = c->nd;
  dh_status st;
  const detham_pt2_options& opt = c->opt;
  const double load = opt.table_load > 0.0 ? fmin(fmax(opt.table_load, 0.05), 0.9) : 0.5;  // target load factor of the HBM table
  // Random 32-byte accesses fall off a cliff once their footprint exceeds what the GPU's TLBs cover: measured on B200,
  // 36 G sectors/s up to 64 GB, 29 at 80 GB, 17 at 96 GB, 8.7 at 160 GB (profiles/r1_microbench.md).  More passes over a
  // smaller table beat fewer passes over a bigger one, so the table never exceeds this many bytes unless configured.
  const double max_table_gb = opt.max_table_gb > 0.0 ? opt.max_table_gb : 60.0;
  // streamed organisation (pt2_stream.cu)
  const bool stream_ok = !ex && opt.mode == 2 && nd >= (int64_t)c->sm_count * 16;

  // a large work space left by expand / ediag would be counted against the table: give it back first
  if (!ex && c->scratch_bytes > ((size_t)256 << 20)) { cudaFree(c->scratch); c->scratch = nullptr; c->scratch_bytes = 0; }

  // ---- plan: partition count and table capacity
  int pbits = 0;
  int64_t slots = opt.table_slots;
  const bool auto_parts = opt.n_parts == 0, auto_slots = slots == 0;
  c->ctr.ms_pt2_plan = 0.0;
  if (!auto_parts) { while ((1 << pbits) < opt.n_parts) ++pbits; }
  int64_t max_slots = slots;
  std::vector<u64> hist;      // class histogram of the contributions (finest partition), empty when nothing was planned
  double hist_scale = 1.0;
  auto max_class = [&](int pb) {  // upper estimate of the contributions of the fullest of 2^pb key partitions
    u64 m = 0;
    for (int cl = 0; cl < (1 << pb); ++cl) { u64 t = 0; for (int f = cl; f < kFine; f += (1 << pb)) t += hist[f]; if (t > m) m = t; }
    return (double)m * hist_scale + 64.0;
  };
  if (auto_parts || auto_slots || stream_ok) {
    // class histogram of the contributions: exact for small inputs, else from every stride-th source (scaled, +10 %);
    // it only sizes the table - an underestimate is caught by the overflow flag and retried with more partitions
    const HbLists* L0 = nullptr;
    st = dh_get_lists(c, 0, &L0); if (st != DH_OK) return st;
    EnumParams P0 = dh_make_params(c, L0);
    const size_t smem = ((dh_cta_table_bytes(c->n) + 15) & ~(size_t)15) + kWarpsPerCta * sizeof(WarpScratch) + kFine * sizeof(unsigned);
    const int64_t stride = nd <= 32768 ? 1 : nd / 16384;
    const int64_t ns = (nd + stride - 1) / stride;
    int64_t want = (ns + kWarpsPerCta - 1) / kWarpsPerCta;
    const int grid = (int)(want < (int64_t)c->sm_count * 4 ? want : (int64_t)c->sm_count * 4);
    DH_CUDA(c, cudaFuncSetAttribute(count_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    DH_CUDA(c, cudaMemsetAsync(c->dcount, 0, 8 * sizeof(u64), c->stream));
    DH_CUDA(c, cudaMemsetAsync(c->hist, 0, kFine * sizeof(u64), c->stream));
    DH_TICK(c, 0);
    count_kernel<false><<<grid, kWarpsPerCta * 32, smem, c->stream>>>(P0, c->dets, psi, nd, stride, eps2, c->dcount, reinterpret_cast<u64*>(c->hist));
    DH_CUDA(c, cudaGetLastError());
    DH_TICK(c, 1);
    hist.assign(kFine, 0);
    DH_CUDA(c, cudaMemcpyAsync(hist.data(), c->hist, kFine * sizeof(u64), cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(c, cudaStreamSynchronize(c->stream));
    c->ctr.ms_pt2_plan = dh_elapsed(c, 0, 1);
    hist_scale = stride == 1 ? 1.0 : 1.1 * (double)stride;
  }
  if (auto_parts || auto_slots) {
    size_t free_b = 0, total_b = 0;
    DH_CUDA(c, cudaMemGetInfo(&free_b, &total_b));
    max_slots = (int64_t)(((double)free_b + (double)c->table_slots * sizeof(Slot) + (double)c->pool_bytes) * 0.92 / sizeof(Slot));
    const int64_t tlb_slots = (int64_t)(max_table_gb * 1e9 / sizeof(Slot));
    if (max_slots > tlb_slots) max_slots = tlb_slots;
    if (!auto_slots) max_slots = slots;
    if (auto_parts) {
      // contributions bound the distinct keys from above; 0.9 of the slots at worst (all distinct) still terminates,
      // and the typical duplication keeps the real load well below that
      pbits = 0;
      while (pbits < DH_MAX_PBITS && max_class(pbits) > 0.9 * (double)max_slots) ++pbits;
      if (max_class(pbits) > 0.9 * (double)max_slots) return DH_ETABLEFULL;
    }
    if (auto_slots) {
      int64_t need = (int64_t)(max_class(pbits) / load) + 1024;
      slots = need < max_slots ? need : max_slots;
    }
  }
  // The streamed organisation runs when asked for (mode 2).  Measured on B200 (profiles/r2_summary.md) it is slower than the
  // table organisation with binned passes on every configuration of BASELINE.json, so the planner does not choose it.
  const bool stream = stream_ok && !hist.empty() && opt.mode == 2;
  int64_t probe_parts = 0;
  double pilot_distinct = 0.0;  // distinct externals of one of 2^pilot_pp key slices
  int pilot_pp = 0;
  if ((auto_parts && auto_slots && pbits >= 3) || stream) {
    // The contribution count bounds the distinct externals from above, often by a wide margin (9 contributions per
    // external on N2-shaped |S| = 1e6), and every pass costs a list start-up per source.  Probe one slice of the key space
    // 8x finer than a planned pass (table organisation), count its distinct keys, and re-plan from that.
    int pp = pbits + 3 < DH_MAX_PBITS ? pbits + 3 : DH_MAX_PBITS;
    int64_t pilot_slots = (pp - pbits == 3 && slots / 4 > 1024) ? slots / 4 : slots;  // 1/8 of the keys in 1/4 of the slots
    if (stream) {  // a slice of about 1e8 contributions: cheap, and still tens of millions of distinct keys
      pp = 0;
      while (pp < DH_MAX_PBITS && max_class(pp) > 1.5e8) ++pp;
      pilot_slots = (int64_t)(max_class(pp) / load) + 1024;
    }
    double pilot[2] = {0.0, 0.0};
    st = pt2_attempt(c, psi, e_s, eps2, pp, pilot_slots, false, load, out, pilot, ex);
    if (c->debug) fprintf(stderr, "[detham] pt2 probe: 1 of %d key slices, %lld slots -> status %d, %.0f distinct, %.1f ms\n", 1 << pp, (long long)pilot_slots, (int)st, pilot[0], pilot[1]);
    if (st == DH_OK) probe_parts = 1ll << pp;
    if (st == DH_OK && pilot[0] > 0.0) {
      c->ctr.ms_pt2_plan += pilot[1];
      pilot_distinct = pilot[0]; pilot_pp = pp;
      if (auto_parts && auto_slots) {
        auto uniq_class = [&](int pb) { const double u = pilot[0] * (double)(1 << (pp - pb)); return 1.2 * u + 8.0 * sqrt(u) + 4096.0; };
        int pb2 = 0;
        while (pb2 < pbits && uniq_class(pb2) > load * (double)max_slots) ++pb2;
        pbits = pb2;
        int64_t need = (int64_t)(uniq_class(pbits) / load);
        // beyond that size the passes run binned and the probes stay in L2, where longer chains cost little while every slot less is 64
        // bytes of DRAM traffic less per pass (fetch + scan): measured on Cr2-shaped, load 0.5 / 0.6 / 0.7 / 0.8: accumulate 5999 /
        // 6004 / 6202 / 6527 ms, scan 810 / 679 / 591 / 534 ms
        if (opt.table_load <= 0.0 && opt.table_regions >= 0 && need * (int64_t)sizeof(Slot) > kBinnedTableBytes) {
          const int64_t denser = (int64_t)(uniq_class(pbits) / 0.6);
          if (denser * (int64_t)sizeof(Slot) > kBinnedTableBytes) need = denser;
        }
        slots = need < max_slots ? need : max_slots;
        if (slots < 1024) slots = 1024;
      }
    } else if (st != DH_OK && st != DH_ETABLEFULL) {
      return st;
    }
  }
  if (stream) {
    // passes: one pass's records (32 bytes each, with head room) must fit the pool budget
    if (c->table) { cudaFree(c->table); c->table = nullptr; c->table_slots = 0; }  // the pilot's table
    size_t free_b = 0, total_b = 0;
    DH_CUDA(c, cudaMemGetInfo(&free_b, &total_b));
    const double budget = opt.stream_pool_gb > 0.0 ? opt.stream_pool_gb * 1e9 : 0.80 * ((double)free_b + (double)c->pool_bytes);
    int sp = 0;
    if (!auto_parts) { while ((1 << sp) < opt.n_parts) ++sp; }
    else while (sp < 8 && max_class(sp) * 1.25 * (double)sizeof(Slot) > budget) ++sp;
    double dscale = 1.15, boost = 1.0;
    for (int tries = 0; tries < 6; ++tries) {
      const double recs = max_class(sp);
      double distinct = pilot_distinct > 0.0 ? fmin(recs, dscale * pilot_distinct * ldexp(1.0, pilot_pp - sp)) : recs;
      const StreamPlan plan{sp, recs * boost, distinct};
      st = dh_pt2_stream(c, psi, e_s, eps2, plan, out);
      if (c->debug) fprintf(stderr, "[detham] pt2 streamed: %d passes, %.3g records and %.3g distinct keys per pass planned (pool budget %.1f GB) -> status %d\n", 1 << sp, recs, distinct, budget / 1e9, (int)st);
      if (st == DH_OK) { c->ctr.pt2_probe_parts = probe_parts; return st; }
      if (st != DH_ETABLEFULL) break;  // DH_EINVAL / DH_ENOMEM: not a case for this organisation
      const bool can_grow = distinct < recs || opt.stream_pool_frac <= 0.0 || (auto_parts && sp < 8);
      if (!can_grow) break;  // nothing left to change: the same attempt would fail the same way
      if (distinct < recs) dscale *= 2.0;   // a region table filled up: the slice probed was not representative
      // a pool segment filled up (the sources a CTA happens to take differ from run to run; with few sources per CTA one CTA can
      // get well over its share): more head room, and more passes where the planner may choose them
      if (opt.stream_pool_frac <= 0.0) boost *= 1.5;  // a configured head room is taken at its word
      if (auto_parts && sp < 8) ++sp;
    }
    if (st != DH_ETABLEFULL && st != DH_EINVAL && st != DH_ENOMEM) return st;
    if (opt.mode == 2) return st;  // asked for explicitly: report instead of switching organisation
    if (c->pool) { cudaFree(c->pool); c->pool = nullptr; c->pool_bytes = 0; }  // make room for the table
  }
  // A plan whose table is beyond kBinnedTableBytes runs binned passes if the record pool of a pass fits beside the table.  Where it does not
  // (many contributions per external: the large N2-shaped sweep points, 9 per external, 4 passes of 6e9 records), more passes of
  // fewer records do, with a smaller table each: measured 20.5-21 G contributions/s binned against 18-19 G/s direct.
  bool force_binned = false;
  if (auto_parts && auto_slots && !ex && !hist.empty() && pilot_distinct > 0.0 && opt.table_regions == 0 &&
      slots * (int64_t)sizeof(Slot) > kBinnedTableBytes) {
    size_t free_b = 0, total_b = 0;
    DH_CUDA(c, cudaMemGetInfo(&free_b, &total_b));
    const double avail = 0.9 * ((double)free_b + (double)c->table_slots * sizeof(Slot) + (double)c->pool_bytes);
    auto uniq = [&](int pb) { const double u = pilot_distinct * ldexp(1.0, pilot_pp - pb); return 1.2 * u + 8.0 * sqrt(u) + 4096.0; };
    auto need_bytes = [&](int pb, double ld) { return (max_class(pb) * 1.2 + 64.0 * 2048 * c->sm_count + uniq(pb) / ld) * (double)sizeof(Slot); };
    if (need_bytes(pbits, 0.6) > avail) {
      for (int pb = pbits + 1; pb <= pbits + 3 && pb <= DH_MAX_PBITS; ++pb)
        if (need_bytes(pb, 0.6) <= avail) {
          pbits = pb;
          slots = (int64_t)(uniq(pb) / 0.6);
          if (slots < 1024) slots = 1024;
          force_binned = true;
          break;
        }
    }
  }
  for (;;) {
    if (ex) DH_CUDA(c, cudaMemsetAsync(ex->cursor, 0, sizeof(u64), c->stream));
    const double est_pass = hist.empty() ? 0.0 : max_class(pbits);  // sizes the record pool of the binned passes
    st = pt2_attempt(c, psi, e_s, eps2, pbits, slots, auto_slots && !ex, load, out, nullptr, ex, est_pass, force_binned);
    if (st == DH_OK) c->ctr.pt2_probe_parts = probe_parts;
    if (st != DH_ETABLEFULL || !auto_parts || pbits >= DH_MAX_PBITS) return st;
    ++pbits;  // the plan was too optimistic: halve the keys per pass and start over
    if (auto_slots) slots = max_slots;
    force_binned = false;
  }
}

// Exact size of the screened connection lists, summed over the sources: an input property (it does not depend on how ham_build
// or pt2 go about their work), the numerator of the benchmark's elements/s.
dh_status dh_count_screened(detham_ctx* c, const double* psi, double thr, int64_t* n_out) {
  const HbLists* L0 = nullptr;
  dh_status st = dh_get_lists(c, 0, &L0); if (st != DH_OK) return st;
  EnumParams P0 = dh_make_params(c, L0);
  const size_t smem = ((dh_cta_table_bytes(c->n) + 15) & ~(size_t)15) + kWarpsPerCta * sizeof(WarpScratch) + kFine * sizeof(unsigned);
  int64_t want = (c->nd + kWarpsPerCta - 1) / kWarpsPerCta;
  const int grid = (int)(want < (int64_t)c->sm_count * 4 ? want : (int64_t)c->sm_count * 4);
  DH_CUDA(c, cudaFuncSetAttribute(count_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  DH_CUDA(c, cudaMemsetAsync(c->dcount, 0, 8 * sizeof(u64), c->stream));
  DH_CUDA(c, cudaMemsetAsync(c->hist, 0, kFine * sizeof(u64), c->stream));
  count_kernel<true><<<grid, kWarpsPerCta * 32, smem, c->stream>>>(P0, c->dets, psi, c->nd, 1, thr, c->dcount, reinterpret_cast<u64*>(c->hist));
  DH_CUDA(c, cudaGetLastError());
  std::vector<u64> hist(kFine);
  DH_CUDA(c, cudaMemcpyAsync(hist.data(), c->hist, kFine * sizeof(u64), cudaMemcpyDeviceToHost, c->stream));
  DH_CUDA(c, cudaStreamSynchronize(c->stream));
  u64 n = 0;
  for (u64 x : hist) n += x;
  *n_out = (int64_t)n;
  return DH_OK;
}

dh_status dh_pt2(detham_ctx* c, const double* psi, double e_s, double eps2, double* out) {
  return pt2_run(c, psi, e_s, eps2, out, nullptr);
}

size_t dh_sort_work_bytes(int64_t m);  // expand.cu
dh_status dh_sort_externals(detham_ctx* c, u64* keys_tmp, double* v_tmp, double* score_tmp, int64_t m, u64* keys_out, double* v_out,
                            double* score_out, void* work);  // expand.cu

// Subspace expansion (row f2): the perturbative set P of Eq. 14 (Alg. 1 "Subspace Expansion"),
// sorted ascending and deduplicated, with score_a = max_i |H_ai psi_i|, v_a = sum_i H_ai psi_i and H_aa.
dh_status dh_expand(detham_ctx* c, const double* psi, double eps2, u64* keys_out, double* score_out, double* v_out, double* haa_out,
                    int64_t cap, int64_t* n_out) {
  u64* cursor = c->dcount + 16;
  // unsorted keys / sums / scores and the sort's buffers live in the context's work space (kept for the next call; detham_trim
  // or a later pt2 that needs the memory releases it)
  const int64_t tcap = cap > 0 ? cap : 1;
  auto al = [](size_t x) { return (x + 255) & ~(size_t)255; };
  const size_t kb = al((size_t)tcap * 2 * sizeof(u64)), vb = v_out ? al((size_t)tcap * sizeof(double)) : 0, sb = score_out ? al((size_t)tcap * sizeof(double)) : 0;
  void* ws = nullptr;
  {
    dh_status st0 = dh_scratch(c, kb + vb + sb + dh_sort_work_bytes(tcap), &ws);
    if (st0 != DH_OK) { cudaGetLastError(); return DH_ENOMEM; }
  }
  char* wp = static_cast<char*>(ws);
  u64* keys_tmp = reinterpret_cast<u64*>(wp);
  double* v_tmp = v_out ? reinterpret_cast<double*>(wp + kb) : nullptr;
  double* score_tmp = score_out ? reinterpret_cast<double*>(wp + kb + vb) : nullptr;
  void* sort_work = wp + kb + vb + sb;
  ExpandOut ex{keys_tmp, v_tmp, score_tmp, (u64)cap, cursor};
  double dummy = 0.0;
  dh_status st = pt2_run(c, psi, 0.0, eps2, &dummy, &ex);
  if (st != DH_OK) return st;
  u64* hp = reinterpret_cast<u64*>(c->pinned);
  DH_CUDA(c, cudaMemcpyAsync(hp, cursor, sizeof(u64), cudaMemcpyDeviceToHost, c->stream));
  DH_CUDA(c, cudaStreamSynchronize(c->stream));
  const int64_t m = (int64_t)hp[0];
  *n_out = m;
  c->ctr.pt2_external = m;
  if (m > cap) return DH_EINVAL;  // *n_out tells the caller how much room it takes
  if (m > 0) {
    st = dh_sort_externals(c, keys_tmp, v_tmp, score_tmp, m, keys_out, v_out, score_out, sort_work);
    if (st == DH_OK && haa_out) st = dh_diagonals(c, keys_out, m, haa_out);
  }
  if (st == DH_OK) DH_CUDA(c, cudaStreamSynchronize(c->stream));
  return st;
}

dh_status dh_connections(detham_ctx* c, int64_t row, double tau, std::vector<u64>& keys, std::vector<double>& h) {
  const HbLists* L = nullptr;
  dh_status st = dh_get_lists(c, 0, &L); if (st != DH_OK) return st;
  EnumParams P = dh_make_params(c, L);
  const int64_t n = c->n, na = c->na, nb = c->nb;
  auto c2 = [](int64_t x) { return x * (x - 1) / 2; };
  int64_t cap = na * (n - na) + nb * (n - nb) + c2(na) * c2(n - na) + c2(nb) * c2(n - nb) + na * nb * (n - na) * (n - nb) + 32;
  void* ws = nullptr;
  st = dh_scratch(c, (size_t)cap * 24 + 256, &ws); if (st != DH_OK) return st;
  u64* dk = static_cast<u64*>(ws);
  double* dh = reinterpret_cast<double*>(dk + 2 * cap);
  int* dn = reinterpret_cast<int*>(dh + cap);
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
  return DH_OK;
}

dh_status dh_diagonals(detham_ctx* c, const u64* dets, int64_t m, double* out) {
  diagonals_kernel<<<(unsigned)((m + 127) / 128), 128, 0, c->stream>>>(c->n, c->J, c->JK, c->hd, c->e_core, dets, m, out);
  DH_CUDA(c, cudaGetLastError());
  return DH_OK;
}
