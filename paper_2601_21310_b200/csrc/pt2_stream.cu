// pt2, streamed organisation (a8, a9) for external sets far beyond L2: no hash table in HBM and no scan kernel.
//
// Per key partition (pass):
//   pt2_gen_kernel    one persistent CTA per SM.  Warps walk the kept prefixes of the heat-bath lists of their sources
//                     (Eq. 14 / the tau rule) and stage every screened, non-member double excitation as an
//                     8-byte reference {list entry, (i,j), source slot, bin}.  When the staging buffer is full the CTA sorts
//                     the references by bin (counting sort: the rank inside the bin comes from the shared-memory counter at
//                     staging time), expands them in bin order into 32-byte records {key, H_ai psi_i, H_aa} (Slater-Condon
//                     value + phase, a5; O(1) diagonal update) and writes each bin's run with consecutive threads into
//                     the CTA's private segment of that bin: whole lines leave the SM, not scattered sectors.
//   pt2_merge_kernel  cooperative launch, one CTA per SM.  Bin b = the externals whose partition word falls into region b.
//                     All warps insert the records of bin b into region table b mod 4 (128-bit CAS claim + fp64 RED, both
//                     served by L2: the four tables are the only memory the kernel addresses by key), then reduce
//                     v_a^2 / (E_S - H_aa) over region b-2 and clear it (Eq. 13 second term).  Warps hand over
//                     through two counters per bin; nothing is written back to HBM but four doubles per CTA.
//
// Members of S are dropped by the generator (membership filter + index of the determinant store, a1), so a record is a
// contribution to an external.  Singles (reading Q5) are evaluated by the walker and written straight into their segment.
#include <stdio.h>
#include <stdlib.h>

#include <algorithm>

#include "pt2_common.cuh"

EnumParams dh_make_params(detham_ctx* c, const HbLists* L);

namespace {

constexpr int kPairChunk = 64;   // occupied pairs per phase-A chunk
constexpr int kMaxSrcSlots = 4;  // sources a warp can have staged references of at one time
constexpr int kMaxBins = 4096;
constexpr int kRing = 3;         // region tables in flight: one being merged into, one being reduced, one cleared for the next
constexpr int kLag = 1;          // the reduce units of region g - kLag follow the merge units of region g in the work list
constexpr int kMergeWarps = 8;    // warps per merge CTA = units per block of the ordered work list
constexpr int kMergeCtasPerSm = 4;
constexpr int kUnitRec = 256;    // records of one merge unit (one warp)
constexpr int kUnitSlots = 512;  // table slots of one reduce unit (one warp)
constexpr int kMergeU = 2;       // records a lane has in flight (their CAS round trips overlap)

// ---------------------------------------------------------------------------------------------- shared-memory layout
struct GenLayout {
  unsigned tables, omask, ptab, keys, warp0, warp_stride, occ_off, zq_off, cp_off, pref_off, beg_off, meta_off, sq_off;
  unsigned cnt, used, cv, haa, meta, bin, rank, order, ctrl, total;
};

__host__ __device__ inline unsigned al16(unsigned x) { return (x + 15u) & ~15u; }

// bytes of staging per reference: H_ai psi_i 8, H_aa 8, orbitals + key slot 4, bin 2, rank 2, order 2
constexpr unsigned kRefBytes = 26u;

__host__ __device__ inline GenLayout gen_layout(int n, int pbits, int npairs, int W, int WU, int K, int B, int N) {
  GenLayout L;
  unsigned o = 0;
  L.tables = o; o = al16(o + (unsigned)(n + 128) * 8u);  // h_pp and the key-partition words; J, J-K stay in L2 (read by rows)
  L.omask = o; o = al16(o + 2u * (1u << pbits) * 8u);
  L.ptab = o; o = al16(o + (unsigned)npairs * 2u);
  L.keys = o; o = al16(o + (unsigned)(W * K) * 16u);     // {alpha, beta} of the sources that staged references point to
  unsigned w = 0;
  w = al16(w + (unsigned)(2 * n) * 8u);                  // U vectors of the warp's current source
  L.occ_off = w; w = al16(w + 4u * DH_MAX_ORB);
  L.zq_off = w; w = al16(w + kPairChunk * 8u);
  L.cp_off = w; w = al16(w + kPairChunk * 8u);
  L.pref_off = w; w = al16(w + (kPairChunk + 1) * 4u);
  L.beg_off = w; w = al16(w + kPairChunk * 4u);
  L.meta_off = w; w = al16(w + kPairChunk * 2u);
  L.sq_off = w; w = al16(w + 96u * 2u);
  L.warp_stride = w;
  L.warp0 = o; o += (unsigned)W * w;
  L.cnt = o; o = al16(o + (unsigned)(B + 1) * 4u);
  L.used = o; o = al16(o + (unsigned)B * 4u);
  const unsigned NS = (unsigned)(N + 32 * WU * W);
  L.cv = o; o = al16(o + NS * 8u);
  L.haa = o; o = al16(o + NS * 8u);
  L.meta = o; o = al16(o + NS * 4u);
  L.bin = o; o = al16(o + NS * 2u);
  L.rank = o; o = al16(o + NS * 2u);
  L.order = o; o = al16(o + NS * 2u);
  L.ctrl = o; o = al16(o + 256u);
  L.total = o;
  return L;
}

// staged reference: H_ai psi_i and H_aa (computed by the walker, whose source is in registers), and 4 bytes of orbitals and
// key slot - a 6 | b 6 | i 6 | j 6 | fam 2 | key slot 6 - from which the expansion rebuilds the 128-bit key


// bit t of the result = parity of the electrons of w below orbital t
__device__ __forceinline__ u64 prefix_parity(u64 w) {
  u64 p = w << 1;
  p ^= p << 1; p ^= p << 2; p ^= p << 4; p ^= p << 8; p ^= p << 16; p ^= p << 32;
  return p;
}
// parity of the electrons strictly between orbitals x and y (x != y), from the prefix-parity word
__device__ __forceinline__ unsigned par_between(u64 pp, int x, int y) {
  const int lo = min(x, y), hi = max(x, y);
  return (unsigned)((pp >> hi) ^ (pp >> (lo + 1))) & 1u;
}
// position of the r-th (0-based) set bit of m
__device__ __forceinline__ int nth_set_bit(u64 m, int r) {
  const unsigned lo = (unsigned)m, hi = (unsigned)(m >> 32);
  const int cl = __popc(lo);
  return r < cl ? (int)__fns(lo, 0u, r + 1) : 32 + (int)__fns(hi, 0u, r - cl + 1);
}
__device__ __forceinline__ unsigned strictly_between(int x, int p, int q) { return (x > min(p, q)) & (x < max(p, q)); }

struct GenParams {
  EnumParams E;
  const u64* dets; const double* psi; int64_t nd; double eps2; unsigned pass;
  const unsigned* sbits; u64 sbits_n; const u64* shash_key; const int* shash_idx; u64 shash_cap;
  int nbins; unsigned seg_cap; Slot* pool; unsigned* used_out;  // used_out [nbins][gridDim.x]
  u64* counters;  // [0] next row [1] generated (members included) [2] contributions
  int* overflow;
  int stage_n, nslots, npairs;
  u64* prof;  // debug: per-CTA cycles of the phases [walk (thread 0's own), walk barrier, sort, expand, advance, rounds], or NULL
};

__device__ __forceinline__ int ld_shared_volatile(const int* p) { return *reinterpret_cast<const volatile int*>(p); }

template <int kGenWarps, int kWalkU>
__global__ void __launch_bounds__(kGenWarps * 32, 1) pt2_gen_kernel(GenParams G) {
  extern __shared__ __align__(16) unsigned char smem[];
  const EnumParams& P = G.E;
  const int n = P.n, na = P.na, nb = P.nb;
  const int NP = 1 << P.pbits;
  const unsigned pmask = (unsigned)NP - 1u;
  const int B = G.nbins, N = G.stage_n, K = G.nslots, npairs = G.npairs;
  const GenLayout L = gen_layout(n, P.pbits, npairs, kGenWarps, kWalkU, K, B, N);
  CtaTables T;
  T.J = const_cast<double*>(P.J); T.JK = const_cast<double*>(P.JK);  // global (L2): only the per-source U vectors read them
  T.hd = reinterpret_cast<double*>(smem + L.tables);
  T.Z = reinterpret_cast<u64*>(T.hd + n);
  for (int t = threadIdx.x; t < n; t += blockDim.x) T.hd[t] = P.hd[t];
  for (int t = threadIdx.x; t < 128; t += blockDim.x) T.Z[t] = dh_zword(t);
  u64* omask = reinterpret_cast<u64*>(smem + L.omask);            // [2][NP]: orbitals of spin s whose class word is c
  unsigned short* ptab = reinterpret_cast<unsigned short*>(smem + L.ptab);  // pair q -> fam << 12 | x << 6 | y (positions in occ)
  unsigned* cnt = reinterpret_cast<unsigned*>(smem + L.cnt);
  unsigned* used = reinterpret_cast<unsigned*>(smem + L.used);
  double* scv = reinterpret_cast<double*>(smem + L.cv);      // staged references (structure of arrays)
  double* shaa = reinterpret_cast<double*>(smem + L.haa);
  unsigned* smeta = reinterpret_cast<unsigned*>(smem + L.meta);
  unsigned short* sbin = reinterpret_cast<unsigned short*>(smem + L.bin);
  ulonglong2* keys = reinterpret_cast<ulonglong2*>(smem + L.keys);  // [warp * K + slot]
  unsigned short* rnk = reinterpret_cast<unsigned short*>(smem + L.rank);
  unsigned short* order = reinterpret_cast<unsigned short*>(smem + L.order);
  int* ctrl = reinterpret_cast<int*>(smem + L.ctrl);  // [0] staged references [1] warps out of work [3] singles of this round [4..] scan carries
  const int tid = threadIdx.x, nthr = blockDim.x;
  const int warp = tid >> 5, lane = tid & 31;
  const unsigned lt = (1u << lane) - 1u;
  const unsigned full = 0xffffffffu;
  const int nAA = na * (na - 1) / 2, nBB = nb * (nb - 1) / 2;
  const int NS = N + 32 * kWalkU * kGenWarps;

  for (int t = tid; t < 2 * NP; t += nthr) omask[t] = 0ull;
  for (int t = tid; t <= B; t += nthr) cnt[t] = 0u;
  for (int t = tid; t < B; t += nthr) used[t] = 0u;
  for (int t = tid; t < NS; t += nthr) order[t] = 0xFFFFu;
  if (tid < 16) ctrl[tid] = 0;
  for (int q = tid; q < npairs; q += nthr) {
    unsigned fam, x, y;
    if (q < nAA + nBB) {
      const int t = q < nAA ? q : q - nAA;
      int yy = (int)((1.0f + sqrtf(1.0f + 8.0f * (float)t)) * 0.5f);
      while (yy * (yy - 1) / 2 > t) --yy;
      while ((yy + 1) * yy / 2 <= t) ++yy;
      fam = q < nAA ? 0u : 1u; x = (unsigned)(t - yy * (yy - 1) / 2); y = (unsigned)yy;
    } else {
      const int r = q - nAA - nBB;
      fam = 2u; x = (unsigned)(r / nb); y = (unsigned)(r % nb);
    }
    ptab[q] = (unsigned short)((fam << 12) | (x << 6) | y);
  }
  __syncthreads();
  if (tid < 2 * n) {  // T.Z is staged by dh_cta_stage
    const int s = tid / n, p = tid % n;
    atomicOr(&omask[s * NP + ((unsigned)T.Z[64 * s + p] & pmask)], 1ull << p);
  }
  __syncthreads();

  unsigned char* wb = smem + L.warp0 + (unsigned)warp * L.warp_stride;
  unsigned char (*occ)[DH_MAX_ORB] = reinterpret_cast<unsigned char (*)[DH_MAX_ORB]>(wb + L.occ_off);  // occ[0..1], vir = occ[2..3]
  double* const U = reinterpret_cast<double*>(wb);  // U[s * n + p] of the warp's current source
  u64* zq = reinterpret_cast<u64*>(wb + L.zq_off);
  double* cp = reinterpret_cast<double*>(wb + L.cp_off);  // per pair of the chunk: E(D) - U(i) - U(j)
  int* pref = reinterpret_cast<int*>(wb + L.pref_off);
  int* pbeg = reinterpret_cast<int*>(wb + L.beg_off);
  unsigned short* pmeta = reinterpret_cast<unsigned short*>(wb + L.meta_off);
  unsigned short* sq = reinterpret_cast<unsigned short*>(wb + L.sq_off);
  const size_t seg_stride = (size_t)gridDim.x * G.seg_cap;  // records between the segments of consecutive bins
  Slot* const my_pool = G.pool + (size_t)blockIdx.x * G.seg_cap;

  // walker state (warp-uniform)
  int phase = 0;  // 0 fetch a source, 1 singles, 2 phase A of chunk qb, 3 phase B
  int cur_slot = 0, qb = 0, pcnt = 0, TT = 0, t0 = 0, qcur = 0, sl = 0, sqn = 0;
  bool out_of_rows = false, reported = false;
  u64 da = 0, db = 0, zsrc = 0, ppa = 0, ppb = 0;
  double psi_v = 0.0, tau = 0.0, e0 = 0.0;
  u64 gen_total = 0, contrib_total = 0;

  long long pc0 = 0, pacc[6] = {0, 0, 0, 0, 0, 0};
  for (;;) {
    if (G.prof && tid == 0) pc0 = clock64();
    // =================================================================== walk: stage references until the buffer is full
    unsigned touched = phase != 0 ? (1u << cur_slot) : 0u;  // slots that staged references of this round point into
    while (ld_shared_volatile(&ctrl[0]) + ld_shared_volatile(&ctrl[3]) < N) {
      if (phase == 0) {
        if (out_of_rows) break;
        const unsigned freem = ~touched & ((1u << K) - 1u);
        if (!freem) break;
        u64 row = 0;
        if (lane == 0) row = atomicAdd(G.counters, 1ull);
        row = __shfl_sync(full, row, 0);
        if ((int64_t)row >= G.nd) { out_of_rows = true; break; }
        psi_v = G.psi[row];
        if (psi_v == 0.0) continue;  // reading Q6: a source with zero amplitude generates nothing
        tau = G.eps2 == 0.0 ? 0.0 : __ddiv_rn(G.eps2, fabs(psi_v));
        da = G.dets[2 * row]; db = G.dets[2 * row + 1];
        cur_slot = __ffs(freem) - 1;
        touched |= 1u << cur_slot;
        // occupied / virtual lists
        for (int p = lane; p < n; p += 32) {
          const u64 below = (1ull << p) - 1ull;
          const int ca = __popcll(da & below), cb = __popcll(db & below);
          if ((da >> p) & 1ull) occ[0][ca] = (unsigned char)p; else occ[2][p - ca] = (unsigned char)p;
          if ((db >> p) & 1ull) occ[1][cb] = (unsigned char)p; else occ[3][p - cb] = (unsigned char)p;
        }
        __syncwarp();
        // partition word of the source
        {
          u64 z = 0;
          if (lane < na) z = T.Z[occ[0][lane]];
          if (lane < nb) z ^= T.Z[64 + occ[1][lane]];
          if (lane + 32 < na) z ^= T.Z[occ[0][lane + 32]];
          if (lane + 32 < nb) z ^= T.Z[64 + occ[1][lane + 32]];
          for (int o = 16; o > 0; o >>= 1) z ^= __shfl_xor_sync(full, z, o);
          zsrc = z;
        }
        // U vectors, E(D), prefix parities; the key goes into the slot that this round's references will name
        for (int p = lane; p < n; p += 32) {
          double ua = T.hd[p], ub = T.hd[p];
          // J and J-K are symmetric (bit for bit: one packed integral each way): row q read by consecutive lanes
          // (four rows' loads are issued before the first is added; the additions keep their order)
          for (int s = 0; s < 2; ++s) {
            const int ne = s ? nb : na;
            const double* A = s ? T.J : T.JK;   // what an electron of spin s adds to U_alpha
            const double* Bm = s ? T.JK : T.J;  // ... and to U_beta
            int k = 0;
            for (; k + 4 <= ne; k += 4) {
              double x[4], y[4];
#pragma unroll
              for (int u = 0; u < 4; ++u) { const int q = occ[s][k + u]; x[u] = __ldg(A + q * n + p); y[u] = __ldg(Bm + q * n + p); }
#pragma unroll
              for (int u = 0; u < 4; ++u) { ua += x[u]; ub += y[u]; }
            }
            for (; k < ne; ++k) { const int q = occ[s][k]; ua += __ldg(A + q * n + p); ub += __ldg(Bm + q * n + p); }
          }
          U[p] = ua; U[n + p] = ub;
        }
        __syncwarp();
        {
          double e = 0.0;
          for (int k = lane; k < na; k += 32) { const int p = occ[0][k]; e += T.hd[p] + U[p]; }
          for (int k = lane; k < nb; k += 32) { const int p = occ[1][k]; e += T.hd[p] + U[n + p]; }
          for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(full, e, o);
          e0 = P.e_core + 0.5 * e;
        }
        ppa = prefix_parity(da); ppb = prefix_parity(db);
        if (lane == 0) keys[warp * K + cur_slot] = make_ulonglong2(da, db);
        __syncwarp();
        phase = 1; sl = 0; sqn = 0;
        continue;
      }
      if (phase == 1) {
        // ---- singles: candidates of this pass's class, queued, evaluated 32 at a time, written straight to their segment
        const int nocc = na + nb;
        bool flush = false;
        if (sl < nocc) {
          const int s = sl >= na ? 1 : 0;
          const int i = occ[s][sl - s * na];
          const u64 w = s ? db : da;
          const unsigned tgt = ((unsigned)(zsrc ^ T.Z[64 * s + i]) ^ G.pass) & pmask;
          const u64 m = omask[s * NP + tgt] & ~w;
          const int c = __popcll(m);
          for (int r = lane; r < c; r += 32) sq[sqn + r] = (unsigned short)((s << 12) | (i << 6) | nth_set_bit(m, r));
          __syncwarp();
          sqn += c;
          ++sl;
          flush = sqn >= 32;
        } else {
          flush = sqn > 0;
          if (!flush) { phase = 2; qb = 0; continue; }
        }
        if (flush) {
          const int take = sqn >= 32 ? 32 : sqn;
          bool ok = false;
          u64 ka = da, kb = db;
          double cv = 0.0, haa = 0.0;
          unsigned bin = 0;
          if (lane < take) {
            const unsigned code = sq[sqn - take + lane];
            const int s = (int)(code >> 12), i = (int)((code >> 6) & 63u), a = (int)(code & 63u);
            const u64 w = s ? db : da;
            const double v = dh_single_value_occ(P, occ, w, s, i, a);
            if (v != 0.0 && fabs(v) >= tau) {
              const u64 nw = (w ^ (1ull << i)) | (1ull << a);
              if (s == 0) ka = nw; else kb = nw;
              const u64 z = zsrc ^ T.Z[64 * s + i] ^ T.Z[64 * s + a];
              ok = true;
              haa = e0 - U[s * n + i] + U[s * n + a] - __ldg(T.JK + i * n + a);
              cv = v * psi_v;
              bin = __umulhi((unsigned)(z >> 32), (unsigned)B);
              // member of S?  (filter first: one 4-byte load settles > 98 % of the non-members)
              bool member = false;
              if (dh_maybe_member(G.sbits, G.sbits_n, z)) member = dh_shash_find(G.shash_key, G.shash_idx, G.shash_cap, ka, kb, z) >= 0;
              gen_total += 1;
              if (member) ok = false;
            }
          }
          __syncwarp();
          sqn -= take;
          const unsigned mk = __ballot_sync(full, ok);
          if (lane == 0 && mk) atomicAdd(&ctrl[3], __popc(mk));
          if (ok) {
            contrib_total += 1;
            const unsigned pos = used[bin] + atomicAdd(&cnt[bin], 1u);
            if (pos < G.seg_cap) dh_st256(my_pool + (size_t)bin * seg_stride + pos, ka, kb, (u64)__double_as_longlong(cv), (u64)__double_as_longlong(haa));
            else *G.overflow = 1;
          }
        }
        continue;
      }
      if (phase == 2) {
        // ---- phase A: kept prefix (|value| >= tau, value != 0) of the class sub-list of every occupied pair of the chunk
        if (qb >= npairs) { phase = 0; continue; }
        const int qe = min(npairs, qb + kPairChunk);
        int cntp = 0, run = 0;
        for (int q0 = qb; q0 < qe; q0 += 32) {
          const int q = q0 + lane;
          int len = 0, beg = 0;
          unsigned pm = 0;
          u64 zij = 0;
          double cpair = 0.0;
          if (q < qe) {
            const unsigned pt = ptab[q];
            const int fam = (int)(pt >> 12), x = (int)((pt >> 6) & 63u), y = (int)(pt & 63u);
            int i, j, seg;
            if (fam == 0) { i = occ[0][x]; j = occ[0][y]; seg = j * (j - 1) / 2 + i; zij = zsrc ^ T.Z[i] ^ T.Z[j]; }
            else if (fam == 1) { i = occ[1][x]; j = occ[1][y]; seg = P.nss + j * (j - 1) / 2 + i; zij = zsrc ^ T.Z[64 + i] ^ T.Z[64 + j]; }
            else { i = occ[0][x]; j = occ[1][y]; seg = 2 * P.nss + i * n + j; zij = zsrc ^ T.Z[i] ^ T.Z[64 + j]; }
            const unsigned cls = ((unsigned)zij ^ G.pass) & pmask;
            const int64_t so = (int64_t)seg * NP + cls;
            beg = __ldg(P.sub_off + so);
            const int end = __ldg(P.sub_off + so + 1);
            // first index whose |value| < tau (tau == 0: whose value == 0, reading Q8): gallop from the head, then bisect
            int lo = beg, hi = end;  // entries before lo are kept, entries from hi on are not
            {
              // four probes at once (most kept prefixes are short), then gallop on or bisect the bracket
              double pv[4];
#pragma unroll
              for (int u = 0; u < 4; ++u) { const int idx = beg + (1 << u) - 1; pv[u] = idx < end ? fabs(__ldg(P.lval + idx)) : 0.0; }
              bool open_end = true;
#pragma unroll
              for (int u = 0; u < 4; ++u) {
                const int idx = beg + (1 << u) - 1;
                if (open_end && idx < end) {
                  if (pv[u] >= tau && pv[u] != 0.0) lo = idx + 1; else { hi = idx; open_end = false; }
                }
              }
              if (open_end && lo < end) {
                int pos = lo + 7, step = 16;
                for (;;) {
                  if (pos >= end) break;
                  const double av = fabs(__ldg(P.lval + pos));
                  if (!(av >= tau && av != 0.0)) break;
                  lo = pos + 1; pos += step; step <<= 1;
                }
                hi = min(pos, end);
              }
              while (lo < hi) {
                const int mid = (lo + hi) >> 1;
                const double av = fabs(__ldg(P.lval + mid));
                if (av >= tau && av != 0.0) lo = mid + 1; else hi = mid;
              }
            }
            len = lo - beg;
            pm = ((unsigned)fam << 12) | ((unsigned)j << 6) | (unsigned)i;  // same field order as the staged reference
            cpair = e0 - U[(fam == 1 ? n : 0) + i] - U[(fam != 0 ? n : 0) + j];
          }
          const unsigned m = __ballot_sync(full, len > 0);
          int x = len;
#pragma unroll
          for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(full, x, o); if (lane >= o) x += y; }
          const int tot = __shfl_sync(full, x, 31);
          if (len > 0) {
            const int idx = cntp + __popc(m & lt);
            pref[idx] = run + x - len; pbeg[idx] = beg; pmeta[idx] = (unsigned short)pm; zq[idx] = zij; cp[idx] = cpair;
          }
          cntp += __popc(m);
          run += tot;
        }
        if (lane == 0) pref[cntp] = run;
        __syncwarp();
        pcnt = cntp; TT = run; t0 = 0; qcur = 0;
        if (TT == 0) { qb += kPairChunk; continue; }
        phase = 3;
        continue;
      }
      // ---- phase B: kWalkU x 32 entries of the concatenated kept prefixes; stage the valid, non-member ones.  Three steps so
      // that the list loads of all batches, then the filter loads of all batches, are in flight together.  The walker's
      // source is in registers and its list entries are consecutive, so value, sign and H_aa are finished here.
      {
        bool ok[kWalkU];
        int mq[kWalkU];
        unsigned abv[kWalkU];
        double lv[kWalkU], ls[kWalkU];
#pragma unroll
        for (int u = 0; u < kWalkU; ++u) {
          ok[u] = false; mq[u] = 0; abv[u] = 0u; lv[u] = 0.0; ls[u] = 0.0;
          const int tt = t0 + 32 * u;
          if (tt < TT) {  // warp-uniform
            const int pe = (qcur + lane < pcnt) ? pref[qcur + lane + 1] - tt : 0x7fffffff;  // end of pair qcur+lane, relative
            const unsigned bm = __reduce_or_sync(full, pe < 32 ? (1u << pe) : 0u);
            const int adv = __popc(__ballot_sync(full, pe <= 32));
            const int myq = qcur + __popc(bm & ((2u << lane) - 1u));
            qcur += adv;
            const int t = tt + lane;
            if (t < TT) {
              ok[u] = true; mq[u] = myq;
              const int k = pbeg[myq] + (t - pref[myq]);
              abv[u] = __ldg(P.lab + k);
              lv[u] = __ldg(P.lval + k);
              ls[u] = __ldg(P.lstat + k);
            }
          }
        }
        u64 zv[kWalkU], fw[kWalkU];
        unsigned pmv[kWalkU];
#pragma unroll
        for (int u = 0; u < kWalkU; ++u) {
          zv[u] = 0ull; fw[u] = 0ull; pmv[u] = 0u;
          if (ok[u]) {
            const unsigned pm = pmeta[mq[u]];
            const int a = (int)(abv[u] & 0xFFu), b = (int)(abv[u] >> 8);
            const unsigned fam = pm >> 12;
            const unsigned si = fam == 1u, sj = fam != 0u;  // spin of (i, a) and of (j, b)
            const u64 wa = si ? db : da, wb2 = sj ? db : da;
            ok[u] = !(((wa >> a) | (wb2 >> b)) & 1ull);
            if (ok[u]) {
              const u64 z = zq[mq[u]] ^ T.Z[64 * si + a] ^ T.Z[64 * sj + b];
              zv[u] = z; pmv[u] = pm;
              fw[u] = __ldg(reinterpret_cast<const u64*>(G.sbits) + dh_filter_word(G.sbits_n, z));
              // H_aa = E(D) - U(i) - U(j) + U(a) + U(b) + the entry's source-independent part (the O(1) diagonal update)
              ls[u] = cp[mq[u]] + U[si * n + a] + U[sj * n + b] + ls[u];
            }
          }
        }
        unsigned msk[kWalkU];
        int nstage = 0;
#pragma unroll
        for (int u = 0; u < kWalkU; ++u) {
          if (ok[u]) {
            gen_total += 1;
            const unsigned pm = pmv[u], fam = pm >> 12;
            const unsigned si = fam == 1u, sj = fam != 0u;
            const int i = (int)(pm & 63u), j = (int)((pm >> 6) & 63u), a = (int)(abv[u] & 0xFFu), b = (int)(abv[u] >> 8);
            const u64 fm = dh_filter_mask(zv[u]);
            if ((fw[u] & fm) == fm) {  // rare: look the key up in the index of S
              const u64 bia = (1ull << i) | (1ull << a), bjb = (1ull << j) | (1ull << b);
              const u64 ka = da ^ ((si ? 0ull : bia) | (sj ? 0ull : bjb)), kb = db ^ ((si ? bia : 0ull) | (sj ? bjb : 0ull));
              if (dh_shash_find(G.shash_key, G.shash_idx, G.shash_cap, ka, kb, zv[u]) >= 0) ok[u] = false;
            }
            // reading Q1: a same-spin double is a+_a a+_b a_j a_i = (a+_b a_j)(a+_a a_i): phase(i->a on w) * phase(j->b on w with
            // i->a applied); an alpha-beta double is the product of its two single phases
            unsigned par = par_between(si ? ppb : ppa, i, a) ^ par_between(sj ? ppb : ppa, j, b);
            if (fam < 2u) par ^= strictly_between(i, j, b) ^ strictly_between(a, j, b);
            lv[u] = (par ? -lv[u] : lv[u]) * psi_v;
          }
          msk[u] = __ballot_sync(full, ok[u]);
          nstage += __popc(msk[u]);
        }
        if (nstage) {
          int base = 0;
          if (lane == 0) base = atomicAdd(&ctrl[0], nstage);
          base = __shfl_sync(full, base, 0);
#pragma unroll
          for (int u = 0; u < kWalkU; ++u) {
            if (ok[u]) {
              const int idx = base + __popc(msk[u] & lt);
              const unsigned bin = __umulhi((unsigned)(zv[u] >> 32), (unsigned)B);
              scv[idx] = lv[u]; shaa[idx] = ls[u];
              // a 6 | b 6 | i 6 | j 6 | fam 2 | key slot 6   (pmv = fam << 12 | j << 6 | i)
              smeta[idx] = (abv[u] & 0x3Fu) | ((abv[u] >> 8) << 6) | ((pmv[u] & 0x3FFFu) << 12) | ((unsigned)(warp * K + cur_slot) << 26);
              sbin[idx] = (unsigned short)bin;
              rnk[idx] = (unsigned short)atomicAdd(&cnt[bin], 1u);
              contrib_total += 1;
            }
            base += __popc(msk[u]);
          }
        }
        t0 += 32 * kWalkU;
        if (t0 >= TT) { qb += kPairChunk; phase = 2; }
      }
    }
    if (out_of_rows && phase == 0 && !reported) { reported = true; if (lane == 0) atomicAdd(&ctrl[1], 1); }
    if (G.prof && tid == 0) { const long long t = clock64(); pacc[0] += t - pc0; pc0 = t; }
    __syncthreads();
    if (G.prof && tid == 0) { const long long t = clock64(); pacc[1] += t - pc0; pc0 = t; }
    const int staged = ctrl[0];
    const bool all_done = ctrl[1] == kGenWarps;

    // =================================================================== sort: exclusive scan of the bin counters
    {
      // per-thread run of bins, warp scan, carry through shared memory
      const int per = (B + nthr - 1) / nthr;
      const int b0 = tid * per, b1 = min(B, b0 + per);
      unsigned s = 0;
      for (int b = b0; b < b1; ++b) s += cnt[b];
      unsigned x = s;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const unsigned y = __shfl_up_sync(full, x, o); if (lane >= o) x += y; }
      unsigned* wsum = reinterpret_cast<unsigned*>(ctrl + 4);  // [kGenWarps]
      if (lane == 31) wsum[warp] = x;
      __syncthreads();
      unsigned carry = 0;
      for (int w = 0; w < warp; ++w) carry += wsum[w];
      unsigned run = carry + x - s;
      for (int b = b0; b < b1; ++b) { const unsigned c = cnt[b]; cnt[b] = run; run += c; }
      if (tid == nthr - 1) cnt[B] = run;
      __syncthreads();
    }
    const int total = (int)cnt[B];  // references + singles of this round
    for (int idx = tid; idx < staged; idx += nthr) order[cnt[sbin[idx]] + rnk[idx]] = (unsigned short)idx;
    __syncthreads();

    if (G.prof && tid == 0) { const long long t = clock64(); pacc[2] += t - pc0; pc0 = t; }
    // =================================================================== expand in bin order and write the runs
    for (int t = tid; t < total; t += nthr) {
      const unsigned idx = order[t];
      if (idx == 0xFFFFu) continue;  // a single: already written by the walker
      order[t] = 0xFFFFu;
      const unsigned m = smeta[idx], bin = sbin[idx];
      const ulonglong2 src = keys[m >> 26];
      const int a = (int)(m & 63u), b = (int)((m >> 6) & 63u), i = (int)((m >> 12) & 63u), j = (int)((m >> 18) & 63u);
      const unsigned fam = (m >> 24) & 3u;
      // one code path for the three families: fam 0 = alpha-alpha, 1 = beta-beta (i<j -> a<b in one spin), 2 = (i alpha -> a, j beta -> b)
      const unsigned si = fam == 1u, sj = fam != 0u;  // spin of (i, a) and of (j, b)
      const u64 bia = (1ull << i) | (1ull << a), bjb = (1ull << j) | (1ull << b);
      const u64 ka = src.x ^ ((si ? 0ull : bia) | (sj ? 0ull : bjb)), kb = src.y ^ ((si ? bia : 0ull) | (sj ? bjb : 0ull));
      const unsigned pos = used[bin] + ((unsigned)t - cnt[bin]);
      if (pos < G.seg_cap) dh_st256(my_pool + (size_t)bin * seg_stride + pos, ka, kb, (u64)__double_as_longlong(scv[idx]), (u64)__double_as_longlong(shaa[idx]));
      else *G.overflow = 1;
    }
    __syncthreads();
    if (G.prof && tid == 0) { const long long t = clock64(); pacc[3] += t - pc0; pc0 = t; }
    // =================================================================== advance the segment fill levels, reset the round
    {
      const int per = (B + nthr - 1) / nthr;
      const int b0 = tid * per, b1 = min(B, b0 + per);
      unsigned nxt = b0 < B ? cnt[b0] : 0u;
      unsigned add[(kMaxBins + kGenWarps * 32 - 1) / (kGenWarps * 32)];
      for (int b = b0; b < b1; ++b) { const unsigned hi = cnt[b + 1]; add[b - b0] = hi - nxt; nxt = hi; }
      __syncthreads();
      for (int b = b0; b < b1; ++b) { used[b] += add[b - b0]; cnt[b] = 0u; }
      if (tid == 0) { cnt[B] = 0u; ctrl[0] = 0; ctrl[3] = 0; }
    }
    __syncthreads();
    if (G.prof && tid == 0) { const long long t = clock64(); pacc[4] += t - pc0; pacc[5] += 1; }
    if (all_done && total == 0) break;
  }
  if (G.prof && tid == 0) for (int k = 0; k < 6; ++k) G.prof[6 * blockIdx.x + k] = (u64)pacc[k];
  unsigned mx = 0;
  for (int b = tid; b < B; b += nthr) { const unsigned ub = min(used[b], G.seg_cap); G.used_out[(size_t)b * gridDim.x + blockIdx.x] = ub; mx = max(mx, ub); }
  for (int o = 16; o > 0; o >>= 1) mx = max(mx, __shfl_xor_sync(full, mx, o));
  if (lane == 0 && mx) atomicMax(G.counters + 20, (u64)mx);  // fullest segment of the pass: sizes the merge's work list
  u64 g = gen_total, ct = contrib_total;
  for (int o = 16; o > 0; o >>= 1) { g += __shfl_xor_sync(full, g, o); ct += __shfl_xor_sync(full, ct, o); }
  if (lane == 0) {
    if (g) atomicAdd(G.counters + 1, g);
    if (ct) atomicAdd(G.counters + 2, ct);
  }
}

// ---------------------------------------------------------------------------------------------- merge + reduce
struct MergeParams {
  const Slot* pool; const unsigned* used; unsigned seg_cap; int nbins, nseg;
  Slot* ring; unsigned cap;  // kRing tables of cap slots
  unsigned* merged; unsigned* cleared;  // [nbins] arrival counters
  double e_s; int n; const double* J; const double* JK; const double* hd; double e_core; double small_den;
  double* part;  // [gridDim.x][4]: sum, sum_abs, min_den, count
  int* overflow;
  u64* ticket;  // next unit of the ordered work list
  const u64* max_used;  // records of the fullest segment of the pass (written by the generator)
  int ring_n, lag;
};

// L2 eviction policies (createpolicy): the region tables are the only reused lines of the merge - evict_last; the records are
// read once - evict_first.  Measured without them (ncu, round 2): 48 % of the CAS and 40 % of the RED sectors missed L2.
__device__ __forceinline__ u64 l2_policy_evict_last() {
  u64 p;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ u64 l2_policy_evict_first() {
  u64 p;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ void red_add_f64_hint(double* addr, double v, u64 pol) {
  asm volatile("red.relaxed.gpu.global.add.L2::cache_hint.f64 [%0], %1, %2;" ::"l"(addr), "d"(v), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_f64_hint(double* addr, double v, u64 pol) {
  asm volatile("st.relaxed.gpu.global.L2::cache_hint.f64 [%0], %1, %2;" ::"l"(addr), "d"(v), "l"(pol) : "memory");
}
__device__ __forceinline__ void ld256_hint(const void* p, u64& a, u64& b, u64& c, u64& d, u64 pol) {
  asm volatile("ld.relaxed.gpu.global.L2::cache_hint.v4.u64 {%0,%1,%2,%3}, [%4], %5;" : "=l"(a), "=l"(b), "=l"(c), "=l"(d) : "l"(p), "l"(pol) : "memory");
}
__device__ __forceinline__ void ld256_stream(const void* p, u64& a, u64& b, u64& c, u64& d, u64 pol) {
  asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.u64 {%0,%1,%2,%3}, [%4], %5;" : "=l"(a), "=l"(b), "=l"(c), "=l"(d) : "l"(p), "l"(pol) : "memory");
}
__device__ __forceinline__ void st256_zero_hint(void* p, u64 pol) {
  asm volatile("st.relaxed.gpu.global.L2::cache_hint.v4.u64 [%0], {%1,%1,%1,%1}, %2;" ::"l"(p), "l"(0ull), "l"(pol) : "memory");
}

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {
  unsigned v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __noinline__ double diag_cold(int n, const double* J, const double* JK, const double* hd, double e_core, u64 a, u64 b) {
  return dh_diag_from_scratch(n, J, JK, hd, e_core, a, b);
}

// Work of one pass = an ORDERED list of units: for region g = 0, 1, ...: the merge units of region g (kUnitRec records of one
// segment each), then the reduce units of region g - kLag (kUnitSlots slots each).  CTAs take blocks of kMergeWarps consecutive
// units from one global counter (one unit per warp), so at any time the whole GPU works inside a window of about one region
// - the three or four region tables it touches stay in L2 - and a slow warp delays only its own unit.  A merge unit of region g
// needs region g - kRing reduced and cleared (same table), a reduce unit of region g needs region g merged: both depend on
// units handed out earlier, to warps that are running (cooperative launch), so the waits cannot deadlock.
__global__ void __launch_bounds__(kMergeWarps * 32, kMergeCtasPerSm) pt2_merge_kernel(MergeParams M) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned full = 0xffffffffu;
  const u64 keep = l2_policy_evict_last(), once = l2_policy_evict_first();
  const unsigned QS = max(1u, ((unsigned)*M.max_used + kUnitRec - 1) / kUnitRec);               // merge units per segment (fullest one)
  const unsigned UM = ((unsigned)M.nseg * QS + kMergeWarps - 1) / kMergeWarps * kMergeWarps;   // merge units per region, whole blocks
  const unsigned US = ((M.cap + kUnitSlots - 1) / kUnitSlots + kMergeWarps - 1) / kMergeWarps * kMergeWarps;  // reduce units per region
  const unsigned GS = UM + US;
  const int kR = M.ring_n, kL = M.lag;
  const u64 total = (u64)(M.nbins + kL) * GS;
  double sum = 0.0, sabs = 0.0, mden = INFINITY, cntd = 0.0;
  __shared__ u64 s_base;
  u64 next = 0;
  if (threadIdx.x == 0) next = atomicAdd(M.ticket, (u64)kMergeWarps);
  for (;;) {
    __syncthreads();  // the previous block's units are done (every warp's atomics issued), s_base may be overwritten
    if (threadIdx.x == 0) s_base = next;
    __syncthreads();
    const u64 base = s_base;
    if (base >= total) break;
    const unsigned g = (unsigned)(base / GS), r = (unsigned)(base % GS);
    const bool is_merge = r < UM;
    const int bin = is_merge ? (int)g : (int)g - kL;
    const bool valid = bin >= 0 && bin < M.nbins;
    if (threadIdx.x == 0) {
      next = atomicAdd(M.ticket, (u64)kMergeWarps);  // the next block's ticket travels while this one is worked on
      if (valid) {
        const unsigned* dep = nullptr;
        unsigned target = 0;
        if (is_merge) { if (bin >= kR) { dep = M.cleared + (bin - kR); target = US / kMergeWarps; } }
        else { dep = M.merged + bin; target = UM / kMergeWarps; }
        if (dep) { unsigned ns = 32; while (ld_acquire_u32(dep) < target) { __nanosleep(ns); if (ns < 1024) ns *= 2; } }
      }
    }
    __syncthreads();
    if (!valid) continue;
    Slot* tb = M.ring + (size_t)(bin % kR) * M.cap;
    if (is_merge) {
      const unsigned u = r + warp;
      const unsigned s = u / QS, q = u % QS;
      if (s < (unsigned)M.nseg) {
        const unsigned nrec = M.used[(size_t)bin * M.nseg + s];
        const unsigned lo = q * kUnitRec, hi = min(nrec, lo + kUnitRec);
        const Slot* src = M.pool + ((size_t)bin * M.nseg + s) * M.seg_cap;
        for (unsigned t0 = lo + lane; t0 < hi; t0 += 32 * kMergeU) {
          u64 ka[kMergeU], kb[kMergeU], vv[kMergeU], hh[kMergeU];
          unsigned slot[kMergeU];
          unsigned pend = 0u;
#pragma unroll
          for (int k = 0; k < kMergeU; ++k) {
            ka[k] = kb[k] = vv[k] = hh[k] = 0ull; slot[k] = 0u;
            const unsigned t = t0 + 32 * k;
            if (t < hi) { ld256_stream(src + t, ka[k], kb[k], vv[k], hh[k], once); pend |= 1u << k; }
          }
#pragma unroll
          for (int k = 0; k < kMergeU; ++k) slot[k] = __umulhi(dh_key_hash(ka[k], kb[k]), M.cap);
          // every pending record's claim is issued before any result is looked at
          for (int probes = 0; pend; ++probes) {
            Key128 old[kMergeU];
#pragma unroll
            for (int k = 0; k < kMergeU; ++k)
              if ((pend >> k) & 1u) old[k] = dh_cas128(tb + slot[k], Key128{0ull, 0ull}, Key128{ka[k], kb[k]});
#pragma unroll
            for (int k = 0; k < kMergeU; ++k)
              if ((pend >> k) & 1u) {
                DH_CHECK(slot[k] < M.cap);
                Slot* sp = tb + slot[k];
                if ((old[k].a | old[k].b) == 0ull) {  // claimed: this thread also records H_aa
                  st_f64_hint(&sp->haa, __longlong_as_double((long long)hh[k]), keep);
                  red_add_f64_hint(&sp->v, __longlong_as_double((long long)vv[k]), keep);
                  pend &= ~(1u << k);
                } else if (old[k].a == ka[k] && old[k].b == kb[k]) {
                  red_add_f64_hint(&sp->v, __longlong_as_double((long long)vv[k]), keep);
                  pend &= ~(1u << k);
                } else if (++slot[k] == M.cap) {
                  slot[k] = 0u;
                }
              }
            if (probes > kProbeLimit) { *M.overflow = 1; break; }
          }
        }
      }
    } else {
      const unsigned u = r - UM + warp;
      const unsigned s_lo = min(M.cap, u * kUnitSlots), s_hi = min(M.cap, s_lo + kUnitSlots);
      constexpr int V = 4;
      for (unsigned t0 = s_lo + lane; t0 < s_hi; t0 += 32 * V) {
        u64 x[V], y[V], z[V], w[V];
#pragma unroll
        for (int k = 0; k < V; ++k) {
          x[k] = y[k] = z[k] = w[k] = 0ull;
          const unsigned t = t0 + 32 * k;
          if (t < s_hi) ld256_hint(tb + t, x[k], y[k], z[k], w[k], keep);
        }
#pragma unroll
        for (int k = 0; k < V; ++k) {
          if (x[k] | y[k]) {
            const double v = __longlong_as_double((long long)z[k]);
            double den = M.e_s - __longlong_as_double((long long)w[k]);
            // H_aa came from the O(1) update of whichever source claimed the slot: where the denominator is small enough to
            // amplify that rounding, take H_aa from the key alone (the same value for every run and partitioning)
            if (fabs(den) < M.small_den) den = M.e_s - diag_cold(M.n, M.J, M.JK, M.hd, M.e_core, x[k], y[k]);
            const double term = v * v / den;
            sum += term; sabs += fabs(term); mden = fmin(mden, fabs(den)); cntd += 1.0;
            st256_zero_hint(tb + t0 + 32 * k, keep);
          }
        }
      }
    }
    __syncthreads();  // every warp of the block has issued its stores and atomics; one release for all of them
    if (threadIdx.x == 0) { __threadfence(); atomicAdd(is_merge ? M.merged + bin : M.cleared + bin, 1u); }
  }
  __shared__ double sh[4][kMergeWarps];
  for (int o = 16; o > 0; o >>= 1) {
    sum += __shfl_xor_sync(full, sum, o); sabs += __shfl_xor_sync(full, sabs, o);
    mden = fmin(mden, __shfl_xor_sync(full, mden, o)); cntd += __shfl_xor_sync(full, cntd, o);
  }
  if (lane == 0) { sh[0][warp] = sum; sh[1][warp] = sabs; sh[2][warp] = mden; sh[3][warp] = cntd; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0, b2 = 0, m = INFINITY, c = 0;
    for (int w = 0; w < kMergeWarps; ++w) { a += sh[0][w]; b2 += sh[1][w]; m = fmin(m, sh[2][w]); c += sh[3][w]; }
    double* o = M.part + 4 * (size_t)blockIdx.x;
    o[0] = a; o[1] = b2; o[2] = m; o[3] = c;
  }
}

__global__ void stream_norm2_kernel(const double* __restrict__ psi, int64_t nd, double* __restrict__ part) {
  double a = 0.0;
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < nd; t += (int64_t)gridDim.x * blockDim.x) a = fma(psi[t], psi[t], a);
  __shared__ double sh[8];
  for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = a;
  __syncthreads();
  if (threadIdx.x == 0) {
    double s = 0;
    for (int w = 0; w < 8; ++w) s += sh[w];
    part[4 * blockIdx.x] = s; part[4 * blockIdx.x + 1] = 0; part[4 * blockIdx.x + 2] = INFINITY; part[4 * blockIdx.x + 3] = 0;
  }
}

}  // namespace

dh_status dh_pt2_stream(detham_ctx* c, const double* psi, double e_s, double eps2, const StreamPlan& plan, double* out) {
  const int64_t nd = c->nd;
  const int n = c->n, na = c->na, nb = c->nb;
  const int pbits = plan.pbits, nparts = 1 << pbits;
  const HbLists* L = nullptr;
  dh_status st = dh_get_lists(c, pbits, &L); if (st != DH_OK) return st;
  GenParams G{};
  G.E = dh_make_params(c, L);
  const int grid = c->sm_count;
  // generator launch shape: 16 warps per CTA, two batches of 32 list entries in flight per warp (24 x 2, 32 x 2 and 32 x 1 were
  // measured too: slower, the staging arrays of 32 warps spill)
  using GenKernel = void (*)(GenParams);
  struct GenVariant { int warps, u; GenKernel k; };
  static const GenVariant variants[] = {{16, 2, pt2_gen_kernel<16, 2>}};
  const int vi = 0;
  const int kGenWarps = variants[vi].warps, kWalkU = variants[vi].u;
  if (nd < (int64_t)grid * kGenWarps || pbits > 8) return DH_EINVAL;  // the caller keeps small inputs on the table organisation

  // ---- region tables: kRing of them share the L2 budget; bins so that a region's distinct keys load it to <= `load`
  const double load = c->opt.stream_load > 0.0 ? c->opt.stream_load : 0.45;
  const double ring_mb = c->opt.stream_ring_mb > 0.0 ? c->opt.stream_ring_mb : 96.0;
  const int ring_n = kRing;
  const double cap_max = ring_mb * 1048576.0 / (ring_n * sizeof(Slot));
  const double distinct = plan.est_distinct > 0.0 ? plan.est_distinct : plan.est_records;
  int nbins = c->opt.stream_bins > 0 ? c->opt.stream_bins : (int)ceil(distinct / (load * cap_max));
  nbins = std::max(nbins, 16);
  if (nbins > kMaxBins) return DH_ETABLEFULL;  // more key partitions needed
  // a region holds its share of the distinct keys plus their spread (hash-uniform bins: 6 sigma) at the target load
  const double per_bin = distinct / nbins;
  const unsigned cap = (unsigned)std::min(4.0e9, std::max(4096.0, (per_bin + 6.0 * sqrt(per_bin) + 64.0) / load));
  const size_t ring_bytes = (size_t)ring_n * cap * sizeof(Slot);
  if (c->ring_bytes < ring_bytes) {
    if (c->ring) cudaFree(c->ring);
    c->ring = nullptr; c->ring_bytes = 0;
    DH_CUDA(c, cudaMalloc(&c->ring, ring_bytes));
    c->ring_bytes = ring_bytes;
  }
  DH_CUDA(c, cudaMemsetAsync(c->ring, 0, ring_bytes, c->stream));  // a failed attempt may have left keys behind

  // ---- record pool: one private segment per (bin, generator CTA)
  const double pool_frac = c->opt.stream_pool_frac > 0.0 ? c->opt.stream_pool_frac : 1.15;
  const double per_seg = plan.est_records / ((double)nbins * grid);
  const unsigned seg_cap = (unsigned)(per_seg * pool_frac + 8.0 * sqrt(per_seg) + 64.0);
  const size_t pool_bytes = (size_t)nbins * grid * seg_cap * sizeof(Slot);
  if ((size_t)c->pool_bytes < pool_bytes) {
    if (c->pool) cudaFree(c->pool);
    c->pool = nullptr; c->pool_bytes = 0;
    size_t free_b = 0, total_b = 0;
    DH_CUDA(c, cudaMemGetInfo(&free_b, &total_b));
    if ((double)pool_bytes > 0.97 * (double)free_b) return DH_ENOMEM;
    if (cudaMalloc(&c->pool, pool_bytes) != cudaSuccess) { cudaGetLastError(); return DH_ENOMEM; }
    c->pool_bytes = (int64_t)pool_bytes;
  }
  const size_t used_bytes = ((size_t)nbins * grid + 2 * (size_t)nbins) * sizeof(unsigned);
  if (c->sflags_bytes < used_bytes) {
    if (c->sflags) cudaFree(c->sflags);
    c->sflags = nullptr; c->sflags_bytes = 0;
    DH_CUDA(c, cudaMalloc(&c->sflags, used_bytes));
    c->sflags_bytes = used_bytes;
  }
  unsigned* used = reinterpret_cast<unsigned*>(c->sflags);
  unsigned* flags = used + (size_t)nbins * grid;

  if (c->debug) fprintf(stderr, "[detham] streamed layout: %d regions of %u slots (%.1f MB ring), segments of %u records, pool %.1f GB\n", nbins, cap, ring_bytes / 1048576.0, seg_cap, pool_bytes / 1e9);
  // ---- generator launch shape: staging takes what the tables and the per-warp scratch leave of the CTA's shared memory
  const int npairs = na * (na - 1) / 2 + nb * (nb - 1) / 2 + na * nb;
  int smem_max = 0;
  DH_CUDA(c, cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, c->device));
  const int K = std::min(kMaxSrcSlots, 64 / kGenWarps);  // key slots per warp (16 bytes each; 6 bits name a slot)
  const GenLayout L0 = gen_layout(n, pbits, npairs, kGenWarps, kWalkU, K, nbins, 0);
  int N = ((int)smem_max - (int)L0.total - 96) / (int)kRefBytes;
  N = std::min(N, 60000) & ~31;
  if (N < 1024) return DH_EINVAL;
  const GenLayout GL = gen_layout(n, pbits, npairs, kGenWarps, kWalkU, K, nbins, N);
  if (c->debug) fprintf(stderr, "[detham] generator: staging %d references, %d source slots per warp, %u bytes of shared memory\n", N, K, GL.total);
  DH_CUDA(c, cudaFuncSetAttribute(variants[vi].k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)GL.total));
  G.dets = c->dets; G.psi = psi; G.nd = nd; G.eps2 = eps2;
  G.sbits = c->sbits; G.sbits_n = (u64)c->sbits_n; G.shash_key = c->shash_key; G.shash_idx = c->shash_idx; G.shash_cap = (u64)c->shash_cap;
  G.nbins = nbins; G.seg_cap = seg_cap; G.pool = reinterpret_cast<Slot*>(c->pool); G.used_out = used;
  G.counters = c->dcount; G.overflow = reinterpret_cast<int*>(c->dcount + 8);
  G.stage_n = N; G.nslots = K; G.npairs = npairs;
  G.prof = nullptr;
  if (c->debug) { DH_CUDA(c, cudaMalloc(&G.prof, 6 * sizeof(u64) * grid)); }

  MergeParams M{};
  M.pool = reinterpret_cast<const Slot*>(c->pool); M.used = used; M.seg_cap = seg_cap; M.nbins = nbins; M.nseg = grid;
  M.ring = reinterpret_cast<Slot*>(c->ring); M.cap = cap; M.merged = flags; M.cleared = flags + nbins;
  M.e_s = e_s; M.n = n; M.J = c->J; M.JK = c->JK; M.hd = c->hd; M.e_core = c->e_core;
  M.small_den = c->opt.small_den == 0.0 ? 1e-3 : (c->opt.small_den < 0.0 ? 0.0 : c->opt.small_den);
  M.overflow = G.overflow;
  M.ticket = c->dcount + 16;
  M.max_used = c->dcount + 20;
  M.ring_n = kRing; M.lag = kLag;
  int merge_occ = 0;
  DH_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&merge_occ, pt2_merge_kernel, kMergeWarps * 32, 0));
  if (merge_occ < 1) return DH_ECUDA;
  const int mgrid = c->sm_count * std::min(merge_occ, kMergeCtasPerSm);  // every CTA resident (cooperative launch): the waits cannot stall

  st = dh_ensure_red(c, 4 * ((int64_t)mgrid + 64) + 4 * (int64_t)(nparts + 1)); if (st != DH_OK) return st;
  double* results = c->red;  // [nparts + 1][4]; row nparts = psi^T psi
  double* part = c->red + 4 * (int64_t)(nparts + 1);
  M.part = part;
  u64* hp = reinterpret_cast<u64*>(c->pinned);
  DH_CUDA(c, cudaMemsetAsync(c->dcount, 0, 32 * sizeof(u64), c->stream));
  stream_norm2_kernel<<<64, 256, 0, c->stream>>>(psi, nd, part);
  dh_launch_final_reduce4(part, 64, results + 4 * nparts, c->stream);
  DH_CUDA(c, cudaGetLastError());

  // The region tables are the merge's only reused lines.  Its loads, stores and reductions carry an evict_last policy; the
  // 128-bit CAS takes no cache hint in PTX (ptxas: "Illegal modifier '.L2::cache_hint' for instruction 'atom'" for cas), so the
  // tables are also declared a persisting access-policy window of the stream for the duration of the call.
  size_t persist_bytes = 0, persist_before = 0;
  cudaStreamAttrValue win_before{};
  {
    int max_persist = 0, max_window = 0;
    DH_CUDA(c, cudaDeviceGetAttribute(&max_persist, cudaDevAttrMaxPersistingL2CacheSize, c->device));
    DH_CUDA(c, cudaDeviceGetAttribute(&max_window, cudaDevAttrMaxAccessPolicyWindowSize, c->device));
    DH_CUDA(c, cudaDeviceGetLimit(&persist_before, cudaLimitPersistingL2CacheSize));
    if (max_persist > 0 && max_window > 0) {
      persist_bytes = std::min(ring_bytes, std::min((size_t)max_persist, (size_t)max_window));
      if (cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, persist_bytes) != cudaSuccess) { cudaGetLastError(); persist_bytes = 0; }
    }
    if (persist_bytes) {
      cudaStreamGetAttribute(c->stream, cudaStreamAttributeAccessPolicyWindow, &win_before);
      cudaStreamAttrValue w{};
      w.accessPolicyWindow.base_ptr = c->ring;
      w.accessPolicyWindow.num_bytes = persist_bytes;
      w.accessPolicyWindow.hitRatio = 1.0f;
      w.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
      w.accessPolicyWindow.missProp = cudaAccessPropertyStreaming;
      if (cudaStreamSetAttribute(c->stream, cudaStreamAttributeAccessPolicyWindow, &w) != cudaSuccess) { cudaGetLastError(); persist_bytes = 0; }
    }
    if (c->debug) fprintf(stderr, "[detham] L2 persistence: device allows %d bytes (window %d), region tables %zu, using %zu\n", max_persist, max_window, ring_bytes, persist_bytes);
  }
  // events: [3 * pass + 0] before gen, +1 between, +2 after merge
  while ((int)c->sev.size() < 3 * nparts) { cudaEvent_t e; DH_CUDA(c, cudaEventCreate(&e)); c->sev.push_back(e); }
  for (int pass = 0; pass < nparts; ++pass) {
    DH_CUDA(c, cudaMemsetAsync(c->dcount, 0, sizeof(u64), c->stream));  // the row cursor; [1], [2], [8] accumulate over the passes
    DH_CUDA(c, cudaMemsetAsync(c->dcount + 16, 0, 8 * sizeof(u64), c->stream));  // the merge's unit counter [16], fullest segment [20]
    DH_CUDA(c, cudaMemsetAsync(flags, 0, 2 * (size_t)nbins * sizeof(unsigned), c->stream));
    DH_CUDA(c, cudaEventRecord(c->sev[3 * pass], c->stream));
    G.pass = (unsigned)pass;
    variants[vi].k<<<grid, kGenWarps * 32, GL.total, c->stream>>>(G);
    DH_CUDA(c, cudaGetLastError());
    DH_CUDA(c, cudaEventRecord(c->sev[3 * pass + 1], c->stream));
    {
      cudaLaunchConfig_t cfg{};
      cfg.gridDim = dim3(mgrid); cfg.blockDim = dim3(kMergeWarps * 32); cfg.dynamicSmemBytes = 0; cfg.stream = c->stream;
      cudaLaunchAttribute at[1];
      at[0].id = cudaLaunchAttributeCooperative; at[0].val.cooperative = 1;
      const unsigned nat = 1;
      cfg.attrs = at; cfg.numAttrs = nat;
      DH_CUDA(c, cudaLaunchKernelEx(&cfg, pt2_merge_kernel, M));
    }
    dh_launch_final_reduce4(part, mgrid, results + 4 * pass, c->stream);
    DH_CUDA(c, cudaGetLastError());
    DH_CUDA(c, cudaEventRecord(c->sev[3 * pass + 2], c->stream));
  }
  if (persist_bytes) {
    DH_CUDA(c, cudaStreamSynchronize(c->stream));
    cudaStreamSetAttribute(c->stream, cudaStreamAttributeAccessPolicyWindow, &win_before);
    cudaCtxResetPersistingL2Cache();
    cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, persist_before);
  }
  if (G.prof) {  // phase cycles of the last pass, averaged over the CTAs
    std::vector<u64> hpf(6 * (size_t)grid);
    DH_CUDA(c, cudaMemcpy(hpf.data(), G.prof, hpf.size() * sizeof(u64), cudaMemcpyDeviceToHost));
    double a[6] = {0, 0, 0, 0, 0, 0};
    for (int b = 0; b < grid; ++b) for (int k = 0; k < 6; ++k) a[k] += (double)hpf[6 * b + k] / grid;
    fprintf(stderr, "[detham] generator phases (cycles per CTA, last pass): walk %.3g, wait for the slowest walker %.3g, sort %.3g, expand %.3g, advance %.3g; %.0f rounds\n", a[0], a[1], a[2], a[3], a[4], a[5]);
    cudaFree(G.prof);
  }
  std::vector<double> res(4 * (size_t)(nparts + 1));
  DH_CUDA(c, cudaMemcpyAsync(res.data(), results, res.size() * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  DH_CUDA(c, cudaMemcpyAsync(hp, c->dcount, 16 * sizeof(u64), cudaMemcpyDeviceToHost, c->stream));
  DH_CUDA(c, cudaStreamSynchronize(c->stream));
  if (*reinterpret_cast<int*>(hp + 8)) return DH_ETABLEFULL;
  double ms_gen = 0.0, ms_merge = 0.0;
  for (int pass = 0; pass < nparts; ++pass) {
    float a = 0.f, b = 0.f;
    cudaEventElapsedTime(&a, c->sev[3 * pass], c->sev[3 * pass + 1]);
    cudaEventElapsedTime(&b, c->sev[3 * pass + 1], c->sev[3 * pass + 2]);
    ms_gen += a; ms_merge += b;
  }
  const double norm2 = res[4 * (size_t)nparts];
  if (!(norm2 > 0.0) || !isfinite(norm2)) return DH_EINVAL;  // psi identically zero (or not finite): Eq. 13 has no value
  double sum = 0, sabs = 0, mden = INFINITY, cnt = 0;
  c->partials.assign(nparts, 0.0);
  for (int p = 0; p < nparts; ++p) {
    c->partials[p] = res[4 * p] / norm2;
    sum += res[4 * p]; sabs += res[4 * p + 1]; mden = fmin(mden, res[4 * p + 2]); cnt += res[4 * p + 3];
  }
  *out = sum / norm2;
  c->ctr.pt2_generated = (int64_t)hp[1];
  c->ctr.pt2_contrib = (int64_t)hp[2];
  c->ctr.pt2_external = (int64_t)cnt;
  c->ctr.pt2_parts = nparts;
  c->ctr.pt2_max_probe = 0;
  c->ctr.pt2_table_slots = (int64_t)cap;
  c->ctr.pt2_binned = 2;
  c->ctr.pt2_stream_bins = nbins;
  c->ctr.pt2_sum_abs = sabs / norm2;
  c->ctr.pt2_min_abs_den = mden;
  c->ctr.ms_pt2_accum = ms_gen;
  c->ctr.ms_pt2_scan = ms_merge;
  return DH_OK;
}
