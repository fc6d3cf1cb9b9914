// Integral-derived tables: J/K matrices (a2) and the heat-bath lists (a3).
#include "common.cuh"

namespace {

__global__ void jk_kernel(int n, const double* __restrict__ h1, const double* __restrict__ eri, double* J, double* JK,
                          double* hd) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n * n) return;
  int p = t / n, q = t % n;
  double j = dh_eri(eri, p, p, q, q), k = dh_eri(eri, p, q, q, p);
  J[t] = j;
  JK[t] = j - k;
  if (p == q) hd[p] = h1[p * n + p];
}

// order inside a segment: class ascending, |value| descending, (a,b) ascending (reading Q15)
__device__ __forceinline__ bool hb_less(double vx, unsigned mx, double vy, unsigned my) {
  unsigned cx = mx >> 16, cy = my >> 16;
  if (cx != cy) return cx < cy;
  double ax = fabs(vx), ay = fabs(vy);
  if (ax != ay) return ax > ay;
  return (mx & 0xFFFFu) < (my & 0xFFFFu);
}

// One CTA per segment: evaluate the segment's integrals, sort them in shared memory (bitonic, ascending comparators
// only so the virtual padding stays at the tail), write values / (a,b) / class offsets.
__global__ void hb_build_kernel(int n, int pbits, int nss, int Lss, int Los, const double* __restrict__ eri,
                                const double* __restrict__ J, const double* __restrict__ JK,
                                int* __restrict__ sub_off, double* __restrict__ val, unsigned short* __restrict__ ab,
                                double* __restrict__ stat, int N /* padded power of two */) {
  extern __shared__ unsigned char smem_raw[];
  double* sv = reinterpret_cast<double*>(smem_raw);
  unsigned* sm = reinterpret_cast<unsigned*>(sv + N);
  const int seg = blockIdx.x;
  const int P = 1 << pbits;
  const unsigned pmask = P - 1;
  int fam, i, j, L;
  int64_t base;
  if (seg < 2 * nss) {
    fam = seg / nss;
    int s = seg % nss;
    j = 1;
    while (j * (j + 1) / 2 <= s) ++j;  // pair id s = j(j-1)/2 + i, i < j
    i = s - j * (j - 1) / 2;
    L = Lss;
    base = (int64_t)seg * Lss;
  } else {
    fam = 2;
    int s = seg - 2 * nss;
    i = s / n;
    j = s % n;
    L = Los;
    base = (int64_t)2 * nss * Lss + (int64_t)s * Los;
  }
  for (int t = threadIdx.x; t < N; t += blockDim.x) {
    double v = 0.0;
    unsigned m = 0xFFFFFFFFu;
    if (t < L) {
      int a, b;
      if (fam < 2) {
        int y = 1;
        while (y * (y + 1) / 2 <= t) ++y;  // t = y(y-1)/2 + x, x < y, over the n-2 orbitals other than i, j
        int x = t - y * (y - 1) / 2;
        a = x; if (a >= i) ++a; if (a >= j) ++a;
        b = y; if (b >= i) ++b; if (b >= j) ++b;
        v = dh_eri(eri, i, a, j, b) - dh_eri(eri, i, b, j, a);
      } else {
        a = t / (n - 1); if (a >= i) ++a;
        b = t % (n - 1); if (b >= j) ++b;
        v = dh_eri(eri, i, a, j, b);
      }
      u64 z = dh_zword(fam == 1 ? 64 + a : a) ^ dh_zword(fam == 0 ? b : 64 + b);
      m = ((unsigned)(z & pmask) << 16) | (unsigned)a | ((unsigned)b << 8);
    }
    sv[t] = v;
    sm[t] = m;
  }
  __syncthreads();
  for (int k = 2; k <= N; k <<= 1) {
    for (int jj = k >> 1; jj > 0; jj >>= 1) {
      for (int t = threadIdx.x; t < N / 2; t += blockDim.x) {
        int lo, hi;
        if (jj == (k >> 1)) {  // flip step: compare with the mirror inside the k-block
          int blk = t / jj, off = t % jj;
          lo = blk * k + off;
          hi = blk * k + k - 1 - off;
        } else {
          int blk = t / jj, off = t % jj;
          lo = blk * 2 * jj + off;
          hi = lo + jj;
        }
        double vl = sv[lo], vh = sv[hi];
        unsigned ml = sm[lo], mh = sm[hi];
        if (hb_less(vh, mh, vl, ml)) { sv[lo] = vh; sv[hi] = vl; sm[lo] = mh; sm[hi] = ml; }
      }
      __syncthreads();
    }
  }
  for (int t = threadIdx.x; t < L; t += blockDim.x) {
    val[base + t] = sv[t];
    ab[base + t] = (unsigned short)(sm[t] & 0xFFFFu);
    // H_aa of the excited determinant = H_ii - U(i) - U(j) + U(a) + U(b) + this (the U are the source's: enumerate.cuh)
    const int a = (int)(sm[t] & 0xFFu), b = (int)((sm[t] >> 8) & 0xFFu);
    const double* X = fam < 2 ? JK : J;
    stat[base + t] = X[i * n + j] + X[a * n + b] - JK[i * n + a] - JK[j * n + b] - X[i * n + b] - X[j * n + a];
  }
  for (int c = threadIdx.x; c < P; c += blockDim.x) {  // first index whose class >= c
    int lo = 0, hi = L;
    while (lo < hi) {
      int mid = (lo + hi) >> 1;
      if ((sm[mid] >> 16) < (unsigned)c) lo = mid + 1; else hi = mid;
    }
    sub_off[(int64_t)seg * P + c] = (int)(base + lo);
  }
  if (seg == gridDim.x - 1 && threadIdx.x == 0) sub_off[(int64_t)gridDim.x * P] = (int)(base + L);
}

}  // namespace

dh_status dh_build_jk(detham_ctx* c) {
  int n = c->n;
  jk_kernel<<<(n * n + 127) / 128, 128, 0, c->stream>>>(n, c->h1, c->eri, c->J, c->JK, c->hd);
  DH_CUDA(c, cudaGetLastError());
  return DH_OK;
}

dh_status dh_get_lists(detham_ctx* c, int pbits, const HbLists** out) {
  if (pbits < 0 || pbits > DH_MAX_PBITS) return DH_EINVAL;
  HbLists& H = c->lists[pbits];
  if (H.pbits == pbits) { *out = &H; return DH_OK; }
  const int n = c->n;
  const int nss = n * (n - 1) / 2;
  const int Lss = n >= 4 ? (n - 2) * (n - 3) / 2 : 0;
  const int Los = (n - 1) * (n - 1);
  const int nseg = 2 * nss + n * n;
  const int64_t total = (int64_t)2 * nss * Lss + (int64_t)n * n * Los;
  const int P = 1 << pbits;
  DH_CUDA(c, cudaMalloc(&H.sub_off, ((int64_t)nseg * P + 1) * sizeof(int)));
  DH_CUDA(c, cudaMalloc(&H.val, (total > 0 ? total : 1) * sizeof(double)));
  DH_CUDA(c, cudaMalloc(&H.ab, (total > 0 ? total : 1) * sizeof(unsigned short)));
  DH_CUDA(c, cudaMalloc(&H.stat, (total > 0 ? total : 1) * sizeof(double)));
  int Lmax = Lss > Los ? Lss : Los;
  int N = 2;
  while (N < Lmax) N <<= 1;
  size_t smem = (size_t)N * (sizeof(double) + sizeof(unsigned));
  DH_CUDA(c, cudaFuncSetAttribute(hb_build_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  hb_build_kernel<<<nseg, 256, smem, c->stream>>>(n, pbits, nss, Lss, Los, c->eri, c->J, c->JK, H.sub_off, H.val, H.ab, H.stat, N);
  DH_CUDA(c, cudaGetLastError());
  H.pbits = pbits;
  H.nseg = nseg;
  H.total = total;
  *out = &H;
  return DH_OK;
}
