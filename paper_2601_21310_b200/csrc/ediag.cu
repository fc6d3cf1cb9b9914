// E_diag = lambda_min(H_SS) ("diagnostic post-hoc diagonalization energy
// E_diag = lambda_min(H_VV), evaluated on the final selected configurations"; Delta_opt = E_var - E_diag).
// Plain Lanczos on the device CSR: the SpMV is the energy kernel's (a second workload for it), the three-term recurrence
// runs in two small fused kernels, the tridiagonal eigenvalue is found on the host by Sturm bisection.  No
// re-orthogonalisation: ghost copies of converged Ritz values do not move the smallest one.
#include <math.h>

#include <vector>

#include "common.cuh"

dh_status dh_spmv(detham_ctx* c, const double* x, double* y, double* xy_out, double* xx_out);  // energy.cu

namespace {

// w = y - alpha v - beta v_prev, partial sums of w^T w
__global__ void __launch_bounds__(256)
lanczos_update_kernel(const double* __restrict__ y, const double* __restrict__ v, const double* __restrict__ vprev, double alpha,
                      double beta, int64_t nd, double* __restrict__ w, double* __restrict__ part) {
  double s = 0.0;
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < nd; t += (int64_t)gridDim.x * blockDim.x) {
    double x = y[t] - alpha * v[t];
    if (vprev) x -= beta * vprev[t];
    w[t] = x;
    s = fma(x, x, s);
  }
  __shared__ double sh[8];
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) { double a = 0; for (int k = 0; k < 8; ++k) a += sh[k]; part[2 * blockIdx.x] = a; part[2 * blockIdx.x + 1] = 0.0; }
}

__global__ void __launch_bounds__(256)
scale_kernel(const double* __restrict__ x, double s, int64_t nd, double* __restrict__ out) {
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < nd; t += (int64_t)gridDim.x * blockDim.x) out[t] = x[t] * s;
}

__global__ void fill_kernel(double* x, double value, int64_t nd) {
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < nd; t += (int64_t)gridDim.x * blockDim.x) x[t] = value;
}

__global__ void sum2_kernel(const double* __restrict__ part, int nblk, double* out) {
  __shared__ double sa[256];
  double a = 0.0;
  for (int t = threadIdx.x; t < nblk; t += 256) a += part[2 * t];
  sa[threadIdx.x] = a;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) { if (threadIdx.x < s) sa[threadIdx.x] += sa[threadIdx.x + s]; __syncthreads(); }
  if (threadIdx.x == 0) out[0] = sa[0];
}

// number of eigenvalues of the symmetric tridiagonal (a, b) below x (Sturm sequence)
int sturm_count(const std::vector<double>& a, const std::vector<double>& b, double x) {
  int cnt = 0;
  double d = 1.0;
  for (size_t k = 0; k < a.size(); ++k) {
    const double off = k == 0 ? 0.0 : b[k - 1] * b[k - 1];
    d = a[k] - x - (k == 0 ? 0.0 : off / d);
    if (d == 0.0) d = -1e-300;
    if (d < 0.0) ++cnt;
  }
  return cnt;
}

// smallest eigenvalue of the tridiagonal; `upper` (if finite) is a known upper bound of it - the previous step's value, since
// the smallest Ritz value never increases from one Lanczos step to the next (Cauchy interlacing)
double tridiag_min(const std::vector<double>& a, const std::vector<double>& b, double upper) {
  double lo = INFINITY, hi = -INFINITY;
  for (size_t k = 0; k < a.size(); ++k) {  // Gershgorin
    const double r = (k > 0 ? fabs(b[k - 1]) : 0.0) + (k + 1 < a.size() ? fabs(b[k]) : 0.0);
    lo = fmin(lo, a[k] - r); hi = fmax(hi, a[k] + r);
  }
  if (isfinite(upper) && upper < hi && upper > lo && sturm_count(a, b, upper) >= 1) hi = upper;
  for (int it = 0; it < 200 && hi - lo > 4e-16 * fmax(fabs(lo), fabs(hi)); ++it) {
    const double mid = 0.5 * (lo + hi);
    if (sturm_count(a, b, mid) >= 1) hi = mid; else lo = mid;
  }
  return 0.5 * (lo + hi);
}

// |last component| of the normalised eigenvector of the tridiagonal for its eigenvalue theta, by the twisted factorisation:
// with the pivots of T - theta I taken from the top (dp) and from the bottom (dm), gamma_r = dp_r + dm_r - (a_r - theta) is
// smallest where the eigenvector is largest; from z_r = 1 the components follow downwards through dp and upwards through dm, both
// in the stable direction.  (A plain top-down pivot sequence meets its near-zero pivot wherever the vector is large - at
// convergence that is far from the last component - and everything after it is wrong.)  beta_k times this number is the residual
// norm ||H y - theta y|| of the Ritz vector y.
double ritz_last_component(const std::vector<double>& a, const std::vector<double>& b, double theta) {
  const int k = (int)a.size();
  if (k == 1) return 1.0;
  std::vector<double> dp(k), dm(k), z(k);
  for (int j = 0; j < k; ++j) {
    dp[j] = a[j] - theta - (j == 0 ? 0.0 : b[j - 1] * b[j - 1] / dp[j - 1]);
    if (dp[j] == 0.0) dp[j] = 1e-300;
  }
  for (int j = k - 1; j >= 0; --j) {
    dm[j] = a[j] - theta - (j == k - 1 ? 0.0 : b[j] * b[j] / dm[j + 1]);
    if (dm[j] == 0.0) dm[j] = 1e-300;
  }
  int r = 0;
  double best = INFINITY;
  for (int j = 0; j < k; ++j) {
    const double g = fabs(dp[j] + dm[j] - (a[j] - theta));
    if (g < best) { best = g; r = j; }
  }
  z[r] = 1.0;
  for (int j = r - 1; j >= 0; --j) z[j] = -b[j] * z[j + 1] / dp[j];
  for (int j = r; j < k - 1; ++j) z[j + 1] = -b[j] * z[j] / dm[j + 1];
  double norm2 = 0.0;
  for (int j = 0; j < k; ++j) norm2 += z[j] * z[j];
  return fabs(z[k - 1]) / sqrt(norm2);
}

}  // namespace

// Stopping rule: with r_k = beta_k |s_k| the residual norm of the smallest Ritz pair (theta_k, y_k), an eigenvalue of H_SS lies
// within r_k of theta_k.  The iteration stops when r_k <= tol |theta_k|, or when the Krylov space closes (beta_k ~ 0: exact);
// otherwise max_iter is reached and *converged_out = 0.  A rule on the movement of theta alone (the first version) takes a start
// vector close to an excited eigenvector for convergence: theta then stagnates for tens of steps while the ground-state
// component grows from rounding level, but r_k stays above the bound all the while.  The price is about twice the steps, since
// theta itself converges like r_k^2 / gap.
dh_status dh_ediag(detham_ctx* c, const double* v0, double tol, int max_iter, double* e_out, int* iters_out, double* resid_out,
                   int* converged_out) {
  const int64_t nd = c->nd;
  const int grid = (int)((nd + 255) / 256 < (int64_t)c->sm_count * 8 ? (nd + 255) / 256 : (int64_t)c->sm_count * 8);
  // v_prev, v, w, y and the partial sums, in the context's work space (no allocation from the second call on)
  void* ws = nullptr;
  dh_status st = dh_scratch(c, ((size_t)4 * nd + 2 * grid + 2) * sizeof(double), &ws); if (st != DH_OK) return st;
  double* buf = static_cast<double*>(ws);
  double* part = buf + 4 * nd;
  double *vprev = buf, *v = buf + nd, *w = buf + 2 * nd, *y = buf + 3 * nd;
  double* h = reinterpret_cast<double*>(c->pinned);
  auto norm2_of = [&](const double* x, double* out) -> dh_status {  // x^T x through the update kernel's reduction (alpha = beta = 0)
    lanczos_update_kernel<<<grid, 256, 0, c->stream>>>(x, x, nullptr, 0.0, 0.0, nd, w, part);
    sum2_kernel<<<1, 256, 0, c->stream>>>(part, grid, part + 2 * grid);
    DH_CUDA(c, cudaGetLastError());
    DH_CUDA(c, cudaMemcpyAsync(h, part + 2 * grid, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(c, cudaStreamSynchronize(c->stream));
    *out = h[0];
    return DH_OK;
  };
  // start vector: the caller's (e.g. psi: already close to the ground vector of H_SS), else all ones
  if (v0) DH_CUDA(c, cudaMemcpyAsync(y, v0, nd * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
  else fill_kernel<<<grid, 256, 0, c->stream>>>(y, 1.0, nd);
  double n2 = 0.0;
  st = norm2_of(y, &n2); if (st != DH_OK) return st;
  if (!(n2 > 0.0) || !isfinite(n2)) return DH_EINVAL;
  scale_kernel<<<grid, 256, 0, c->stream>>>(y, 1.0 / sqrt(n2), nd, v);
  std::vector<double> a, b;
  double beta = 0.0, theta = 0.0, theta_prev = INFINITY, resid = INFINITY;
  int it = 0, converged = 0;
  for (; it < max_iter; ++it) {
    double alpha = 0.0, vv = 0.0;
    st = dh_spmv(c, v, y, &alpha, &vv); if (st != DH_OK) return st;  // alpha = v^T H v (v is normalised)
    alpha /= vv;
    a.push_back(alpha);
    theta = tridiag_min(a, b, theta_prev);
    lanczos_update_kernel<<<grid, 256, 0, c->stream>>>(y, v, it > 0 ? vprev : nullptr, alpha, beta, nd, w, part);
    sum2_kernel<<<1, 256, 0, c->stream>>>(part, grid, part + 2 * grid);
    DH_CUDA(c, cudaGetLastError());
    DH_CUDA(c, cudaMemcpyAsync(h, part + 2 * grid, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(c, cudaStreamSynchronize(c->stream));
    beta = sqrt(h[0]);
    const double scale = fmax(fabs(theta), 1e-300);
    if (!(beta > 1e-14 * fmax(fabs(alpha), 1.0))) { resid = beta; converged = 1; ++it; break; }  // invariant subspace: theta is exact
    resid = beta * ritz_last_component(a, b, theta);
    theta_prev = theta;
    if (resid <= tol * scale) { converged = 1; ++it; break; }
    b.push_back(beta);
    double* t = vprev; vprev = v; v = t;           // v_prev <- v
    scale_kernel<<<grid, 256, 0, c->stream>>>(w, 1.0 / beta, nd, v);  // v <- w / beta
    DH_CUDA(c, cudaGetLastError());
  }
  DH_CUDA(c, cudaStreamSynchronize(c->stream));
  *e_out = theta;
  if (iters_out) *iters_out = it;
  if (resid_out) *resid_out = resid;
  if (converged_out) *converged_out = converged;
  return DH_OK;
}
