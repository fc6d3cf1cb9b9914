// energy (a7): y = H_SS psi fused with psi^T y and psi^T psi (Eq. 11; the SpMV of PAPER.md:282).
#include "common.cuh"

namespace {

// TPR threads cooperate on one row; per-CTA partial sums go to `part` and are reduced in a fixed order afterwards
// so the result is reproducible run to run.
template <int TPR>
__global__ void __launch_bounds__(256)
spmv_energy_kernel(const int64_t* __restrict__ row_ptr, const int* __restrict__ col, const double* __restrict__ val,
                   const double* __restrict__ psi, int64_t nd, double* __restrict__ y_out, double* __restrict__ part) {
  const int sub = threadIdx.x % TPR;
  const int64_t rows_per_cta = 256 / TPR;
  double num = 0.0, den = 0.0;
  for (int64_t rbase = (int64_t)blockIdx.x * rows_per_cta; rbase < nd; rbase += (int64_t)gridDim.x * rows_per_cta) {
    const int64_t row = rbase + threadIdx.x / TPR;  // loop bounds are CTA-uniform so the sub-warp shuffles stay convergent
    const bool live = row < nd;
    const int64_t b = live ? row_ptr[row] : 0, e = live ? row_ptr[row + 1] : 0;
    double acc = 0.0;
    for (int64_t k = b + sub; k < e; k += TPR) { DH_CHECK(col[k] >= 0 && col[k] < nd); acc = fma(val[k], __ldg(psi + col[k]), acc); }
#pragma unroll
    for (int o = TPR / 2; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o, TPR);
    if (sub == 0 && live) {
      double p = psi[row];
      if (y_out) y_out[row] = acc;
      num = fma(p, acc, num);
      den = fma(p, p, den);
    }
  }
  __shared__ double sn[8], sd[8];
  for (int o = 16; o > 0; o >>= 1) { num += __shfl_xor_sync(0xffffffffu, num, o); den += __shfl_xor_sync(0xffffffffu, den, o); }
  if ((threadIdx.x & 31) == 0) { sn[threadIdx.x >> 5] = num; sd[threadIdx.x >> 5] = den; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0.0, b = 0.0;
    for (int w = 0; w < 8; ++w) { a += sn[w]; b += sd[w]; }
    part[2 * blockIdx.x] = a;
    part[2 * blockIdx.x + 1] = b;
  }
}

// residual r = H_SS psi - e psi (the vector Eq. 12 contracts with grad psi) fused with the internal term of
// Eq. 13 (first sum): sum_i r_i^2 / (e - H_ii); H_ii is the row's own diagonal entry.  TPR threads per row,
// chosen like the energy kernel's.
template <int TPR>
__global__ void __launch_bounds__(256)
residual_kernel(const int64_t* __restrict__ row_ptr, const int* __restrict__ col, const double* __restrict__ val,
                const double* __restrict__ psi, int64_t nd, double e, double* __restrict__ r_out, double* __restrict__ part) {
  const int sub = threadIdx.x % TPR;
  const int64_t rows_per_cta = 256 / TPR;
  double num = 0.0, den = 0.0;
  for (int64_t rbase = (int64_t)blockIdx.x * rows_per_cta; rbase < nd; rbase += (int64_t)gridDim.x * rows_per_cta) {
    const int64_t row = rbase + threadIdx.x / TPR;
    const bool live = row < nd;
    const int64_t b = live ? row_ptr[row] : 0, en = live ? row_ptr[row + 1] : 0;
    double acc = 0.0, hii = 0.0;
    for (int64_t k = b + sub; k < en; k += TPR) {
      const int c = col[k];
      const double v = val[k];
      acc = fma(v, __ldg(psi + c), acc);
      if (c == row) hii = v;
    }
#pragma unroll
    for (int o = TPR / 2; o > 0; o >>= 1) {
      acc += __shfl_xor_sync(0xffffffffu, acc, o, TPR);
      hii += __shfl_xor_sync(0xffffffffu, hii, o, TPR);  // exactly one lane holds the diagonal, the others 0
    }
    if (sub == 0 && live) {
      const double p = psi[row];
      const double r = acc - e * p;
      if (r_out) r_out[row] = r;
      if (r != 0.0) num += r * r / (e - hii);
      den = fma(p, p, den);
    }
  }
  __shared__ double sn[8], sd[8];
  for (int o = 16; o > 0; o >>= 1) { num += __shfl_xor_sync(0xffffffffu, num, o); den += __shfl_xor_sync(0xffffffffu, den, o); }
  if ((threadIdx.x & 31) == 0) { sn[threadIdx.x >> 5] = num; sd[threadIdx.x >> 5] = den; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0.0, b2 = 0.0;
    for (int w = 0; w < 8; ++w) { a += sn[w]; b2 += sd[w]; }
    part[2 * blockIdx.x] = a;
    part[2 * blockIdx.x + 1] = b2;
  }
}

__global__ void final_reduce2_kernel(const double* __restrict__ part, int nblk, double* out) {
  __shared__ double sa[256], sb[256];
  double a = 0.0, b = 0.0;
  for (int t = threadIdx.x; t < nblk; t += 256) { a += part[2 * t]; b += part[2 * t + 1]; }
  sa[threadIdx.x] = a; sb[threadIdx.x] = b;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if (threadIdx.x < s) { sa[threadIdx.x] += sa[threadIdx.x + s]; sb[threadIdx.x] += sb[threadIdx.x + s]; }
    __syncthreads();
  }
  if (threadIdx.x == 0) { out[0] = sa[0]; out[1] = sb[0]; }
}

}  // namespace

dh_status dh_ensure_red(detham_ctx* c, int64_t n) {
  if (c->red_cap >= n) return DH_OK;
  if (c->red) cudaFree(c->red);
  c->red = nullptr; c->red_cap = 0;
  DH_CUDA(c, cudaMalloc(&c->red, n * sizeof(double)));
  c->red_cap = n;
  return DH_OK;
}

dh_status dh_scratch(detham_ctx* c, size_t bytes, void** p) {
  if (c->scratch_bytes < bytes) {
    if (c->scratch) cudaFree(c->scratch);
    c->scratch = nullptr; c->scratch_bytes = 0;
    DH_CUDA(c, cudaMalloc(&c->scratch, bytes));
    c->scratch_bytes = bytes;
  }
  *p = c->scratch;
  return DH_OK;
}

dh_status dh_energy(detham_ctx* c, const double* psi, double* e_out, double* n2_out, double* y_out) {
  const int64_t nd = c->nd;
  const double avg = (double)c->nnz / (double)nd;
  const int tpr = avg <= 6 ? 4 : (avg <= 24 ? 8 : 32);
  int64_t want = (nd + (256 / tpr) - 1) / (256 / tpr);
  int grid = (int)(want < (int64_t)c->sm_count * 8 ? want : (int64_t)c->sm_count * 8);
  dh_status st = dh_ensure_red(c, 2 * (int64_t)grid + 2);
  if (st != DH_OK) return st;
  double* part = c->red + 2;
  DH_TICK(c, 0);
  if (tpr == 4) spmv_energy_kernel<4><<<grid, 256, 0, c->stream>>>(c->row_ptr, c->col, c->val, psi, nd, y_out, part);
  else if (tpr == 8) spmv_energy_kernel<8><<<grid, 256, 0, c->stream>>>(c->row_ptr, c->col, c->val, psi, nd, y_out, part);
  else spmv_energy_kernel<32><<<grid, 256, 0, c->stream>>>(c->row_ptr, c->col, c->val, psi, nd, y_out, part);
  DH_CUDA(c, cudaGetLastError());
  final_reduce2_kernel<<<1, 256, 0, c->stream>>>(part, grid, c->red);
  DH_CUDA(c, cudaGetLastError());
  DH_TICK(c, 1);
  double* h = reinterpret_cast<double*>(c->pinned);
  DH_CUDA(c, cudaMemcpyAsync(h, c->red, 2 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  DH_CUDA(c, cudaStreamSynchronize(c->stream));
  c->ctr.ms_energy = dh_elapsed(c, 0, 1);
  if (!(h[1] > 0.0) || !isfinite(h[1])) return DH_EINVAL;  // psi identically zero (or not finite): Eq. 11 has no value
  *e_out = h[0] / h[1];
  if (n2_out) *n2_out = h[1];
  return DH_OK;
}

dh_status dh_residual(detham_ctx* c, const double* psi, double e_s, double* r_out, double* internal_out) {
  const int64_t nd = c->nd;
  const double avg = (double)c->nnz / (double)nd;
  const int tpr = avg <= 6 ? 4 : (avg <= 24 ? 8 : 32);
  int64_t want = (nd + (256 / tpr) - 1) / (256 / tpr);
  int grid = (int)(want < (int64_t)c->sm_count * 8 ? want : (int64_t)c->sm_count * 8);
  dh_status st = dh_ensure_red(c, 2 * (int64_t)grid + 2);
  if (st != DH_OK) return st;
  double* part = c->red + 2;
  if (tpr == 4) residual_kernel<4><<<grid, 256, 0, c->stream>>>(c->row_ptr, c->col, c->val, psi, nd, e_s, r_out, part);
  else if (tpr == 8) residual_kernel<8><<<grid, 256, 0, c->stream>>>(c->row_ptr, c->col, c->val, psi, nd, e_s, r_out, part);
  else residual_kernel<32><<<grid, 256, 0, c->stream>>>(c->row_ptr, c->col, c->val, psi, nd, e_s, r_out, part);
  DH_CUDA(c, cudaGetLastError());
  final_reduce2_kernel<<<1, 256, 0, c->stream>>>(part, grid, c->red);
  DH_CUDA(c, cudaGetLastError());
  double* h = reinterpret_cast<double*>(c->pinned);
  DH_CUDA(c, cudaMemcpyAsync(h, c->red, 2 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  DH_CUDA(c, cudaStreamSynchronize(c->stream));
  *internal_out = h[0] / h[1];
  return DH_OK;
}

// y = H_SS x with x^T y and x^T x (the Lanczos step of ediag.cu); same kernels as dh_energy, no timers
dh_status dh_spmv(detham_ctx* c, const double* x, double* y, double* xy_out, double* xx_out) {
  const int64_t nd = c->nd;
  const double avg = (double)c->nnz / (double)nd;
  const int tpr = avg <= 6 ? 4 : (avg <= 24 ? 8 : 32);
  int64_t want = (nd + (256 / tpr) - 1) / (256 / tpr);
  int grid = (int)(want < (int64_t)c->sm_count * 8 ? want : (int64_t)c->sm_count * 8);
  dh_status st = dh_ensure_red(c, 2 * (int64_t)grid + 2);
  if (st != DH_OK) return st;
  double* part = c->red + 2;
  if (tpr == 4) spmv_energy_kernel<4><<<grid, 256, 0, c->stream>>>(c->row_ptr, c->col, c->val, x, nd, y, part);
  else if (tpr == 8) spmv_energy_kernel<8><<<grid, 256, 0, c->stream>>>(c->row_ptr, c->col, c->val, x, nd, y, part);
  else spmv_energy_kernel<32><<<grid, 256, 0, c->stream>>>(c->row_ptr, c->col, c->val, x, nd, y, part);
  DH_CUDA(c, cudaGetLastError());
  final_reduce2_kernel<<<1, 256, 0, c->stream>>>(part, grid, c->red);
  DH_CUDA(c, cudaGetLastError());
  double* h = reinterpret_cast<double*>(c->pinned) + 8;
  DH_CUDA(c, cudaMemcpyAsync(h, c->red, 2 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  DH_CUDA(c, cudaStreamSynchronize(c->stream));
  *xy_out = h[0];
  *xx_out = h[1];
  return DH_OK;
}
