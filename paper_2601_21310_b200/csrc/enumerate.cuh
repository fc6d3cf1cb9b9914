// Excitation enumeration with early exit (a4) and Slater-Condon value + fermionic phase (a5).
// One warp per source determinant.  PAPER.md:227: "The algorithm iterates through the pre-sorted virtual pairs,
// enabling an 'early exit' once |<ij||ab>| < tau.  Configurations with negligible coupling are thus never generated."
#pragma once
#include "common.cuh"

struct EnumParams {
  int n, na, nb;
  int pbits;                 // lists are split into 1 << pbits key classes
  int nss;                   // n(n-1)/2
  const double* h1;          // [n*n]
  const double* eri;         // packed
  const int* sub_off;        // heat-bath lists
  const double* lval;
  const unsigned short* lab;
  const double* lstat;       // per list entry: source-independent part of the diagonal update (HbLists::stat)
  const double* J;           // global copies staged into shared memory by cta_stage
  const double* JK;
  const double* hd;
  double e_core;
};

// CTA-wide shared tables: J, J-K, h_pp, key-partition words.
struct CtaTables {
  double* J;    // [n*n]
  double* JK;   // [n*n]
  double* hd;   // [n]
  u64* Z;       // [128]
};

// per-warp scratch
struct WarpScratch {
  double U[2][DH_MAX_ORB];          // U_sigma(p) = h_pp + sum_{q in occ_sigma} (J-K)_pq + sum_{q in occ_other} J_pq
  unsigned char occ[2][DH_MAX_ORB];
  unsigned char vir[2][DH_MAX_ORB];
};

__host__ __device__ inline size_t dh_cta_table_bytes(int n) { return (size_t)(2 * n * n + n) * sizeof(double) + 128 * sizeof(u64); }

// kStageJK = false (the pt2 accumulate kernel): J and J-K stay in global memory and are read through L1 - per source they are
// touched by dh_fill_U (the rows of the occupied orbitals: the same ~20 KB for most sources) and by the few singles - which leaves
// 50 KB more of the SM's L1 / shared-memory array to the L1 that serves the heat-bath lists; only h_pp and the Zobrist words are
// staged (dh_cta_light_bytes).
__host__ __device__ inline size_t dh_cta_light_bytes(int n) { return (size_t)n * sizeof(double) + 128 * sizeof(u64); }

template <bool kStageJK = true>
__device__ __forceinline__ CtaTables dh_cta_stage(const EnumParams& P, unsigned char* smem) {
  CtaTables T;
  const int n = P.n;
  if (!kStageJK) {
    T.J = const_cast<double*>(P.J);
    T.JK = const_cast<double*>(P.JK);
    T.hd = reinterpret_cast<double*>(smem);
    T.Z = reinterpret_cast<u64*>(T.hd + n);
    for (int t = threadIdx.x; t < n; t += blockDim.x) T.hd[t] = P.hd[t];
    for (int t = threadIdx.x; t < 128; t += blockDim.x) T.Z[t] = dh_zword(t);
    __syncthreads();
    return T;
  }
  T.J = reinterpret_cast<double*>(smem);
  T.JK = T.J + n * n;
  T.hd = T.JK + n * n;
  T.Z = reinterpret_cast<u64*>(T.hd + n);
  for (int t = threadIdx.x; t < n * n; t += blockDim.x) { T.J[t] = P.J[t]; T.JK[t] = P.JK[t]; }
  for (int t = threadIdx.x; t < n; t += blockDim.x) T.hd[t] = P.hd[t];
  for (int t = threadIdx.x; t < 128; t += blockDim.x) T.Z[t] = dh_zword(t);
  __syncthreads();
  return T;
}

// occupied / virtual orbital lists of both spin strings (ascending), by all lanes of the warp
__device__ __forceinline__ void dh_fill_occ(const EnumParams& P, WarpScratch& ws, u64 da, u64 db, int lane) {
  for (int p = lane; p < P.n; p += 32) {
    u64 below = (1ull << p) - 1ull;
    int ca = __popcll(da & below), cb = __popcll(db & below);
    if ((da >> p) & 1ull) ws.occ[0][ca] = (unsigned char)p; else ws.vir[0][p - ca] = (unsigned char)p;
    if ((db >> p) & 1ull) ws.occ[1][cb] = (unsigned char)p; else ws.vir[1][p - cb] = (unsigned char)p;
  }
  __syncwarp();
}

// U vectors and the source's diagonal E(D) = e_core + 1/2 sum_{p occ} (h_pp + U(p)); returns E(D) on every lane
__device__ __forceinline__ double dh_fill_U(const EnumParams& P, const CtaTables& T, WarpScratch& ws, int lane) {
  const int n = P.n;
  for (int p = lane; p < n; p += 32) {
    double ua = T.hd[p], ub = T.hd[p];
    // J and J-K are symmetric (bit for bit: both triangles come from the same packed integral), so row q is read at column p:
    // the lanes (p = lane) then touch consecutive words instead of words n apart (a 16-way bank conflict at n = 56)
    for (int k = 0; k < P.na; ++k) { int q = ws.occ[0][k]; ua += T.JK[q * n + p]; ub += T.J[q * n + p]; }
    for (int k = 0; k < P.nb; ++k) { int q = ws.occ[1][k]; ua += T.J[q * n + p]; ub += T.JK[q * n + p]; }
    ws.U[0][p] = ua;
    ws.U[1][p] = ub;
  }
  __syncwarp();
  double e = 0.0;
  for (int k = lane; k < P.na; k += 32) { int p = ws.occ[0][k]; e += T.hd[p] + ws.U[0][p]; }
  for (int k = lane; k < P.nb; k += 32) { int p = ws.occ[1][k]; e += T.hd[p] + ws.U[1][p]; }
  for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
  return P.e_core + 0.5 * e;
}

// H_aa of an excited determinant from the source's E(D) and U vectors (O(1) update; differs from a from-scratch sum
// by rounding only, reading Q16).  kind: 0 single in spin s; 1 same-spin double in spin s; 2 alpha-beta double.
__device__ __forceinline__ double dh_excited_diag(const CtaTables& T, const WarpScratch& ws, int n, double e0, int kind,
                                                  int s, int i, int j, int a, int b) {
  if (kind == 0) return e0 - ws.U[s][i] + ws.U[s][a] - T.JK[i * n + a];
  if (kind == 1)
    return e0 - ws.U[s][i] - ws.U[s][j] + ws.U[s][a] + ws.U[s][b] + T.JK[i * n + j] + T.JK[a * n + b] - T.JK[i * n + a] -
           T.JK[i * n + b] - T.JK[j * n + a] - T.JK[j * n + b];
  return e0 - ws.U[0][i] - ws.U[1][j] + ws.U[0][a] + ws.U[1][b] + T.J[i * n + j] + T.J[a * n + b] - T.JK[i * n + a] -
         T.JK[j * n + b] - T.J[i * n + b] - T.J[j * n + a];
}

// Single-excitation element i -> a in spin s, evaluation order of DESIGN.md reading Q7 (adds only, no FMA possible):
// h_ia, then ((ia|qq) - (iq|qa)) over same-spin occupied q ascending, then (ia|qq) over other-spin occupied q ascending.
__device__ __forceinline__ double dh_single_value_occ(const EnumParams& P, const unsigned char (*occ)[DH_MAX_ORB], u64 wsame, int s, int i, int a) {
  double v = __ldg(P.h1 + i * P.n + a);
  const int ns = s == 0 ? P.na : P.nb, no = s == 0 ? P.nb : P.na;
  // the loads of four terms are issued before the first is added (the additions keep the order of reading Q7)
  int k = 0;
  for (; k + 4 <= ns; k += 4) {
    double t[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) { const int q = occ[s][k + u]; t[u] = dh_eri(P.eri, i, a, q, q) - dh_eri(P.eri, i, q, q, a); }
#pragma unroll
    for (int u = 0; u < 4; ++u) v = v + t[u];
  }
  for (; k < ns; ++k) { const int q = occ[s][k]; v = v + (dh_eri(P.eri, i, a, q, q) - dh_eri(P.eri, i, q, q, a)); }
  k = 0;
  for (; k + 4 <= no; k += 4) {
    double t[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) { const int q = occ[s ^ 1][k + u]; t[u] = dh_eri(P.eri, i, a, q, q); }
#pragma unroll
    for (int u = 0; u < 4; ++u) v = v + t[u];
  }
  for (; k < no; ++k) { const int q = occ[s ^ 1][k]; v = v + dh_eri(P.eri, i, a, q, q); }
  return dh_parity_between(wsame, i, a) ? -v : v;
}
__device__ __forceinline__ double dh_single_value(const EnumParams& P, const WarpScratch& ws, u64 wsame, int s, int i, int a) {
  return dh_single_value_occ(P, ws.occ, wsame, s, i, a);
}

// parity (0 even, 1 odd) of the phase of a double excitation of (da, db), reading Q1.  kind 1: same spin s, i<j -> a<b:
// a+_a a+_b a_j a_i = (a+_b a_j)(a+_a a_i): phase(i->a on w) * phase(j->b on w with i->a applied).  kind 2: i alpha -> a,
// j beta -> b: the product of the two single phases.
__device__ __forceinline__ int dh_double_parity(u64 da, u64 db, int kind, int s, int i, int j, int a, int b) {
  if (kind == 1) {
    const u64 w = s ? db : da;
    return dh_parity_between(w, i, a) ^ dh_parity_between((w ^ (1ull << i)) | (1ull << a), j, b);
  }
  return dh_parity_between(da, i, a) ^ dh_parity_between(db, j, b);
}

// Enumerate every excitation D' of (da, db) with |H| >= tau, H != 0 whose key class (low pbits of its partition word)
// equals `pass`, and hand it to the sink.  Requires dh_fill_occ done.  All 32 lanes call sink.emit convergently:
//   sink.emit(active, ka, kb, z, H, kind, s, i, j, a, b)
// If Sink::kLookupFirst, singles are offered to sink.pre(ka, kb, z) before their O(N_e) evaluation.
// If Sink::kLazySign, doubles arrive with the list's value, WITHOUT the fermionic phase: a sink that drops most candidates
// (ham_build: 98 % are not in S) applies dh_double_parity itself to the few it keeps.
template <class Sink>
__device__ __forceinline__ void dh_enumerate(const EnumParams& P, const CtaTables& T, const WarpScratch& ws, u64 da, u64 db,
                                             double tau, u64 zsrc, unsigned pass, Sink& sink, int lane) {
  const int n = P.n;
  const unsigned pmask = (1u << P.pbits) - 1u;
  const int NP = 1 << P.pbits;
  // ---- singles (reading Q5: every single is generated and evaluated exactly)
  for (int s = 0; s < 2; ++s) {
    const int no = s == 0 ? P.na : P.nb, nv = n - no;
    const u64 w = s == 0 ? da : db;
    const int total = no * nv;
    for (int t0 = 0; t0 < total; t0 += 32) {
      int t = t0 + lane;
      bool act = t < total;
      int i = 0, a = 0;
      u64 ka = da, kb = db, z = zsrc;
      double v = 0.0;
      if (act) {
        i = ws.occ[s][t / nv];
        a = ws.vir[s][t % nv];
        u64 nw = (w ^ (1ull << i)) | (1ull << a);
        if (s == 0) ka = nw; else kb = nw;
        z = zsrc ^ T.Z[64 * s + i] ^ T.Z[64 * s + a];
        act = ((unsigned)z & pmask) == pass;
        if (Sink::kLookupFirst && act) act = sink.pre(ka, kb, z);
        if (act) {
          v = dh_single_value(P, ws, w, s, i, a);
          act = (v != 0.0) && (fabs(v) >= tau);
        }
      }
      sink.emit(act, ka, kb, z, v, 0, s, i, 0, a, 0);
    }
  }
  // ---- same-spin doubles: walk the (i<j) list of the wanted class while |<ij||ab>| >= tau
  for (int s = 0; s < 2; ++s) {
    const int no = s == 0 ? P.na : P.nb;
    const u64 w = s == 0 ? da : db;
    for (int jj = 1; jj < no; ++jj) {
      const int j = ws.occ[s][jj];
      for (int ii = 0; ii < jj; ++ii) {
        const int i = ws.occ[s][ii];
        const u64 zij = zsrc ^ T.Z[64 * s + i] ^ T.Z[64 * s + j];
        const unsigned cls = ((unsigned)zij ^ pass) & pmask;
        const int64_t so = (int64_t)(s * P.nss + j * (j - 1) / 2 + i) * NP + cls;
        const int beg = __ldg(P.sub_off + so), end = __ldg(P.sub_off + so + 1);
        const u64 wij = w ^ (1ull << i) ^ (1ull << j);
        // the next 32 entries (value and orbital pair) are loaded before this batch is looked up, so the list latency hides
        // behind the sink's; the batch past the early exit is loaded in vain (one per pair)
        double vn = beg + lane < end ? __ldg(P.lval + beg + lane) : 0.0;
        unsigned mn = beg + lane < end ? __ldg(P.lab + beg + lane) : 0u;
        for (int k0 = beg; k0 < end; k0 += 32) {
          const bool inb = k0 + lane < end;
          double v = vn;
          const unsigned m = mn;
          const int kn = k0 + 32 + lane;
          vn = kn < end ? __ldg(P.lval + kn) : 0.0;
          mn = kn < end ? __ldg(P.lab + kn) : 0u;
          bool big = inb && fabs(v) >= tau;
          bool act = big && v != 0.0;
          int a = 0, b = 0;
          u64 ka = da, kb = db, z = zij;
          if (act) {
            a = m & 0xFF; b = m >> 8;
            act = !((w >> a) & 1ull) && !((w >> b) & 1ull);
            if (act) {
              u64 nw = wij | (1ull << a) | (1ull << b);
              if (s == 0) ka = nw; else kb = nw;
              z = zij ^ T.Z[64 * s + a] ^ T.Z[64 * s + b];
              if (!Sink::kLazySign && dh_double_parity(da, db, 1, s, i, j, a, b)) v = -v;
            }
          }
          sink.emit(act, ka, kb, z, v, 1, s, i, j, a, b);
          if (__ballot_sync(0xffffffffu, big) != 0xffffffffu) break;  // early exit
        }
      }
    }
  }
  // ---- opposite-spin doubles: (i alpha -> a, j beta -> b), value (ia|jb)
  for (int ii = 0; ii < P.na; ++ii) {
    const int i = ws.occ[0][ii];
    for (int jj = 0; jj < P.nb; ++jj) {
      const int j = ws.occ[1][jj];
      const u64 zij = zsrc ^ T.Z[i] ^ T.Z[64 + j];
      const unsigned cls = ((unsigned)zij ^ pass) & pmask;
      const int64_t so = (int64_t)(2 * P.nss + i * n + j) * NP + cls;
      const int beg = __ldg(P.sub_off + so), end = __ldg(P.sub_off + so + 1);
      double vn = beg + lane < end ? __ldg(P.lval + beg + lane) : 0.0;
      unsigned mn = beg + lane < end ? __ldg(P.lab + beg + lane) : 0u;
      for (int k0 = beg; k0 < end; k0 += 32) {
        const bool inb = k0 + lane < end;
        double v = vn;
        const unsigned m = mn;
        const int kn = k0 + 32 + lane;
        vn = kn < end ? __ldg(P.lval + kn) : 0.0;
        mn = kn < end ? __ldg(P.lab + kn) : 0u;
        bool big = inb && fabs(v) >= tau;
        bool act = big && v != 0.0;
        int a = 0, b = 0;
        u64 ka = da, kb = db, z = zij;
        if (act) {
          a = m & 0xFF; b = m >> 8;
          act = !((da >> a) & 1ull) && !((db >> b) & 1ull);
          if (act) {
            ka = (da ^ (1ull << i)) | (1ull << a);
            kb = (db ^ (1ull << j)) | (1ull << b);
            z = zij ^ T.Z[a] ^ T.Z[64 + b];
            if (!Sink::kLazySign && dh_double_parity(da, db, 2, 0, i, j, a, b)) v = -v;
          }
        }
        sink.emit(act, ka, kb, z, v, 2, 0, i, j, a, b);
        if (__ballot_sync(0xffffffffu, big) != 0xffffffffu) break;
      }
    }
  }
}

// partition word of a determinant (XOR over occupied spin-orbitals), one thread
__device__ __forceinline__ u64 dh_zobrist(u64 da, u64 db, const u64* Z) {
  u64 z = 0;
  while (da) { int p = __ffsll((long long)da) - 1; da &= da - 1; z ^= Z[p]; }
  while (db) { int p = __ffsll((long long)db) - 1; db &= db - 1; z ^= Z[64 + p]; }
  return z;
}
