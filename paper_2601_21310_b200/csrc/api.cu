// C ABI entry points (include/detham.h): argument checks, context lifetime, host<->device plumbing.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <numeric>

#include "common.cuh"

namespace {

bool is_device_ptr(const void* p) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}



void free_all(detham_ctx* c) {
  auto f = [](void* p) { if (p) cudaFree(p); };
  f(c->h1); f(c->eri); f(c->J); f(c->JK); f(c->hd);
  for (auto& L : c->lists) { f(L.sub_off); f(L.val); f(L.ab); f(L.stat); }
  f(c->dets_owned); f(c->psi_owned); f(c->shash_key); f(c->shash_idx); f(c->sbits);
  f(c->row_ptr); f(c->col); f(c->val); f(c->row_cnt); f(c->sp_row_ptr); f(c->sp_col); f(c->sp_val); f(c->phash_key); f(c->phash_idx); f(c->acol); f(c->aval); f(c->segs); f(c->table); f(c->pool); f(c->ring); f(c->sflags); f(c->pair_galpha); f(c->pair_gstart); f(c->pair_diag); f(c->pair_akey); f(c->pair_bused); f(c->red); f(c->dcount); f(c->hist); f(c->scratch); f(c->perm);
  if (c->pinned) cudaFreeHost(c->pinned);
  for (auto& e : c->ev) if (e) cudaEventDestroy(e);
  for (auto& e : c->sev) cudaEventDestroy(e);
}

}  // namespace

extern "C" {

dh_status detham_create(detham_ctx** out, int n_orb, int n_alpha, int n_beta, const double* h1, const double* eri,
                        double e_core, void* cuda_stream) {
  if (!out) return DH_EINVAL;
  *out = nullptr;
  if (!h1 || !eri || n_orb < 1 || n_orb > DH_MAX_ORB || n_alpha < 0 || n_beta < 0 || n_alpha > n_orb || n_beta > n_orb ||
      n_alpha + n_beta < 1 || !std::isfinite(e_core))
    return DH_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return DH_ECUDA; }
  detham_ctx* c = new (std::nothrow) detham_ctx;
  if (!c) return DH_ENOMEM;
  c->n = n_orb; c->na = n_alpha; c->nb = n_beta; c->e_core = e_core;
  c->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
  if (const char* e = getenv("DETHAM_DEBUG")) c->debug = e[0] == '1';  // the library's one environment switch
  auto fail = [&](dh_status s) { free_all(c); delete c; return s; };
  auto body = [&]() -> dh_status {
    DH_CUDA(c, cudaGetDevice(&c->device));
    DH_CUDA(c, cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, c->device));
    const int64_t n = n_orb, npair = n * (n + 1) / 2;
    c->n_eri = npair * (npair + 1) / 2;
    DH_CUDA(c, cudaMalloc(&c->h1, n * n * sizeof(double)));
    DH_CUDA(c, cudaMalloc(&c->eri, c->n_eri * sizeof(double)));
    DH_CUDA(c, cudaMalloc(&c->J, n * n * sizeof(double)));
    DH_CUDA(c, cudaMalloc(&c->JK, n * n * sizeof(double)));
    DH_CUDA(c, cudaMalloc(&c->hd, n * sizeof(double)));
    DH_CUDA(c, cudaMalloc(&c->dcount, 64 * sizeof(u64)));
    DH_CUDA(c, cudaMalloc(&c->hist, 1024 * sizeof(int64_t)));
    DH_CUDA(c, cudaMallocHost(&c->pinned, 4096));
    for (auto& e : c->ev) DH_CUDA(c, cudaEventCreate(&e));
    DH_CUDA(c, cudaMemcpyAsync(c->h1, h1, n * n * sizeof(double), is_device_ptr(h1) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, c->stream));
    DH_CUDA(c, cudaMemcpyAsync(c->eri, eri, c->n_eri * sizeof(double), is_device_ptr(eri) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, c->stream));
    dh_status st = dh_build_jk(c);
    if (st != DH_OK) return st;
    const HbLists* L = nullptr;
    st = dh_get_lists(c, 0, &L);
    if (st != DH_OK) return st;
    DH_CUDA(c, cudaStreamSynchronize(c->stream));
    return DH_OK;
  };
  dh_status st = body();
  if (st != DH_OK) return fail(st);
  *out = c;
  return DH_OK;
}

dh_status detham_set_subspace(detham_ctx* c, const uint64_t* dets, int64_t n_dets) {
  if (!c || !dets || n_dets < 1 || n_dets >= (1ll << 31)) return DH_EINVAL;
  if (!is_device_ptr(dets)) return DH_EINVAL;
  c->dets = nullptr; c->nd = 0; c->nnz = -1; c->sp_nnz = -1;
  DH_TICK(c, 0);
  dh_status st = dh_validate_subspace(c, reinterpret_cast<const u64*>(dets), n_dets);
  if (st != DH_OK) return st;
  c->dets = reinterpret_cast<const u64*>(dets);
  c->nd = n_dets;
  st = dh_build_shash(c);
  if (st != DH_OK) return st;
  DH_TICK(c, 1);
  DH_CUDA(c, cudaEventSynchronize(c->ev[1]));
  c->ctr.ms_store = dh_elapsed(c, 0, 1);
  return DH_OK;
}

dh_status detham_ham_build(detham_ctx* c, double eps, int64_t* nnz_out) {
  if (!c || !c->dets || !(eps >= 0.0)) return DH_EINVAL;
  dh_status st = dh_ham_build(c, eps);
  if (st == DH_OK && nnz_out) *nnz_out = c->nnz;
  return st;
}

dh_status detham_build_config(detham_ctx* c, int method) {
  if (!c || method < 0 || method > 2) return DH_EINVAL;
  c->build_method = method;
  return DH_OK;
}

dh_status detham_csr(detham_ctx* c, const int64_t** row_ptr, const int32_t** col, const double** val) {
  if (!c || c->nnz < 0 || !row_ptr || !col || !val) return DH_EINVAL;
  *row_ptr = c->row_ptr; *col = c->col; *val = c->val;
  return DH_OK;
}

dh_status detham_csr_copy(detham_ctx* c, int64_t* row_ptr, int32_t* col, double* val) {
  if (!c || c->nnz < 0) return DH_EINVAL;
  auto kind = [](const void* p) { return is_device_ptr(p) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost; };
  if (row_ptr) DH_CUDA(c, cudaMemcpyAsync(row_ptr, c->row_ptr, (c->nd + 1) * sizeof(int64_t), kind(row_ptr), c->stream));
  if (col && c->nnz) DH_CUDA(c, cudaMemcpyAsync(col, c->col, c->nnz * sizeof(int), kind(col), c->stream));
  if (val && c->nnz) DH_CUDA(c, cudaMemcpyAsync(val, c->val, c->nnz * sizeof(double), kind(val), c->stream));
  DH_CUDA(c, cudaStreamSynchronize(c->stream));
  return DH_OK;
}

dh_status detham_energy(detham_ctx* c, const double* psi, double* e_out, double* norm2_out, double* y_out) {
  if (!c || !psi || !e_out || c->nnz < 0) return DH_EINVAL;
  return dh_energy(c, psi, e_out, norm2_out, y_out);
}

dh_status detham_residual(detham_ctx* c, const double* psi, double e_s, double* r_out, double* internal_out) {
  if (!c || !psi || !internal_out || c->nnz < 0 || !std::isfinite(e_s)) return DH_EINVAL;
  return dh_residual(c, psi, e_s, r_out, internal_out);
}

dh_status detham_ediag(detham_ctx* c, const double* v0, double tol, int max_iter, double* e_out, int* iters_out, double* resid_out,
                       int* converged_out) {
  if (!c || !e_out || c->nnz < 0 || !(tol > 0.0) || max_iter < 1) return DH_EINVAL;
  return dh_ediag(c, v0, tol, max_iter, e_out, iters_out, resid_out, converged_out);
}

dh_status detham_pt2_config(detham_ctx* c, int64_t table_slots, int n_parts) {
  if (!c || table_slots < 0 || n_parts < 0 || n_parts > (1 << DH_MAX_PBITS) || (n_parts & (n_parts - 1))) return DH_EINVAL;
  if (table_slots > 0 && table_slots < 64) return DH_EINVAL;
  c->opt.table_slots = table_slots;
  c->opt.n_parts = n_parts;
  return DH_OK;
}

dh_status detham_pt2_set_options(detham_ctx* c, const detham_pt2_options* o) {
  if (!c) return DH_EINVAL;
  if (!o) { c->opt = detham_pt2_options{}; return DH_OK; }
  auto fin = [](double x) { return std::isfinite(x); };
  if (o->mode < 0 || o->mode > 2 || o->n_parts < 0 || o->n_parts > (1 << DH_MAX_PBITS) || (o->n_parts & (o->n_parts - 1)) ||
      o->table_slots < 0 || (o->table_slots > 0 && o->table_slots < 64) || !fin(o->table_load) || o->table_load < 0.0 ||
      o->table_load > 0.95 || !fin(o->max_table_gb) || o->max_table_gb < 0.0 || !fin(o->small_den) || o->table_regions < -1 || (o->table_regions > 0 && (o->table_regions < 64 || o->table_regions > 8192)) || o->stream_bins < 0 ||
      o->stream_bins > 4096 || !fin(o->stream_ring_mb) || o->stream_ring_mb < 0.0 || !fin(o->stream_load) || o->stream_load < 0.0 ||
      o->stream_load > 0.95 || !fin(o->stream_pool_frac) || o->stream_pool_frac < 0.0 || !fin(o->stream_pool_gb) || o->stream_pool_gb < 0.0)
    return DH_EINVAL;
  c->opt = *o;
  return DH_OK;
}

dh_status detham_trim(detham_ctx* c) {
  if (!c) return DH_EINVAL;
  DH_CUDA(c, cudaStreamSynchronize(c->stream));
  auto f = [](auto*& p) { if (p) cudaFree(p); p = nullptr; };
  f(c->table); c->table_slots = 0;
  f(c->pool); c->pool_bytes = 0;
  f(c->ring); c->ring_bytes = 0;
  f(c->sflags); c->sflags_bytes = 0;
  f(c->scratch); c->scratch_bytes = 0;
  for (int k = 1; k <= DH_MAX_PBITS; ++k) {
    HbLists& L = c->lists[k];
    f(L.sub_off); f(L.val); f(L.ab); f(L.stat);
    L.pbits = -1;
  }
  return DH_OK;
}

dh_status detham_pt2(detham_ctx* c, const double* psi, double e_s, double eps2, double* pt2_out, int64_t* n_external_out,
                     int64_t* n_contrib_out) {
  if (!c || !c->dets || !psi || !pt2_out || !(eps2 >= 0.0) || !std::isfinite(e_s)) return DH_EINVAL;
  dh_status st = dh_pt2(c, psi, e_s, eps2, pt2_out);
  if (st != DH_OK) return st;
  if (n_external_out) *n_external_out = c->ctr.pt2_external;
  if (n_contrib_out) *n_contrib_out = c->ctr.pt2_contrib;
  return DH_OK;
}

dh_status detham_count_screened(detham_ctx* c, const double* psi, double thr, int64_t* n_out) {
  if (!c || !c->dets || !(thr >= 0.0) || !n_out) return DH_EINVAL;
  return dh_count_screened(c, psi, thr, n_out);
}

dh_status detham_expand(detham_ctx* c, const double* psi, double eps2, uint64_t* keys_out, double* score_out, double* v_out,
                        double* haa_out, int64_t cap, int64_t* n_out) {
  if (!c || !c->dets || !psi || !(eps2 >= 0.0) || !n_out || cap < 0 || (cap > 0 && !keys_out)) return DH_EINVAL;
  return dh_expand(c, psi, eps2, reinterpret_cast<u64*>(keys_out), score_out, v_out, haa_out, cap, n_out);
}

dh_status detham_complete_sum(detham_ctx* c, const double* psi, const uint64_t* pkeys, int64_t m, double* v_out) {
  if (!c || !c->dets || !psi || m < 0 || m >= (1ll << 31) || (m > 0 && (!pkeys || !v_out || !is_device_ptr(pkeys)))) return DH_EINVAL;
  return dh_complete_sum(c, psi, reinterpret_cast<const u64*>(pkeys), m, v_out);
}

dh_status detham_hsp_build(detham_ctx* c, const double* psi, double eps2, const uint64_t* pkeys, int64_t m, int64_t* nnz_out) {
  if (!c || !c->dets || !psi || !(eps2 >= 0.0) || m < 0 || m >= (1ll << 31) || (m > 0 && (!pkeys || !is_device_ptr(pkeys)))) return DH_EINVAL;
  c->sp_nnz = -1;
  dh_status st = dh_hsp_build(c, psi, eps2, reinterpret_cast<const u64*>(pkeys), m);
  if (st == DH_OK && nnz_out) *nnz_out = c->sp_nnz;
  return st;
}

dh_status detham_hsp_csr(detham_ctx* c, const int64_t** row_ptr, const int32_t** col, const double** val) {
  if (!c || c->sp_nnz < 0 || !row_ptr || !col || !val) return DH_EINVAL;
  *row_ptr = c->sp_row_ptr; *col = c->sp_col; *val = c->sp_val;
  return DH_OK;
}

dh_status detham_hsp_csr_copy(detham_ctx* c, int64_t* row_ptr, int32_t* col, double* val) {
  if (!c || c->sp_nnz < 0) return DH_EINVAL;
  auto kind = [](const void* p) { return is_device_ptr(p) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost; };
  if (row_ptr) DH_CUDA(c, cudaMemcpyAsync(row_ptr, c->sp_row_ptr, (c->nd + 1) * sizeof(int64_t), kind(row_ptr), c->stream));
  if (col && c->sp_nnz) DH_CUDA(c, cudaMemcpyAsync(col, c->sp_col, c->sp_nnz * sizeof(int), kind(col), c->stream));
  if (val && c->sp_nnz) DH_CUDA(c, cudaMemcpyAsync(val, c->sp_val, c->sp_nnz * sizeof(double), kind(val), c->stream));
  DH_CUDA(c, cudaStreamSynchronize(c->stream));
  return DH_OK;
}

dh_status detham_pt2_partials(detham_ctx* c, double* out, int cap, int* n_parts_out) {
  if (!c || !out || cap < 0) return DH_EINVAL;
  int m = (int)c->partials.size();
  if (n_parts_out) *n_parts_out = m;
  for (int k = 0; k < m && k < cap; ++k) out[k] = c->partials[k];
  return DH_OK;
}

dh_status detham_solve_host(detham_ctx* c, const uint64_t* dets_host, const double* psi_host, int64_t n_dets, double eps,
                            double eps2, double* e_out, double* pt2_out, int64_t* nnz_out, int64_t* n_external_out) {
  if (!c || !dets_host || !psi_host || n_dets < 1 || n_dets >= (1ll << 31) || !e_out || !pt2_out) return DH_EINVAL;
  if (!(eps >= 0.0) || !(eps2 >= 0.0)) return DH_EINVAL;
  if (c->owned_cap < n_dets) {
    if (c->dets_owned) cudaFree(c->dets_owned);
    if (c->psi_owned) cudaFree(c->psi_owned);
    c->dets_owned = nullptr; c->psi_owned = nullptr; c->owned_cap = 0;
    DH_CUDA(c, cudaMalloc(&c->dets_owned, n_dets * 2 * sizeof(u64)));
    DH_CUDA(c, cudaMalloc(&c->psi_owned, n_dets * sizeof(double)));
    c->owned_cap = n_dets;
  }
  DH_CUDA(c, cudaMemcpyAsync(c->dets_owned, dets_host, n_dets * 2 * sizeof(u64), cudaMemcpyHostToDevice, c->stream));
  DH_CUDA(c, cudaMemcpyAsync(c->psi_owned, psi_host, n_dets * sizeof(double), cudaMemcpyHostToDevice, c->stream));
  dh_status st = detham_set_subspace(c, reinterpret_cast<const uint64_t*>(c->dets_owned), n_dets);
  if (st != DH_OK) return st;
  st = detham_ham_build(c, eps, nnz_out);
  if (st != DH_OK) return st;
  double norm2 = 0.0;
  st = detham_energy(c, c->psi_owned, e_out, &norm2, nullptr);
  if (st != DH_OK) return st;
  return detham_pt2(c, c->psi_owned, *e_out, eps2, pt2_out, n_external_out, nullptr);
}

dh_status detham_connections(detham_ctx* c, int64_t row, double tau, uint64_t* keys_out, double* h_out, int64_t cap,
                             int64_t* n_out) {
  if (!c || !c->dets || row < 0 || row >= c->nd || !(tau >= 0.0) || !n_out || cap < 0) return DH_EINVAL;
  std::vector<u64> keys; std::vector<double> h;
  dh_status st = dh_connections(c, row, tau, keys, h);
  if (st != DH_OK) return st;
  const int64_t m = (int64_t)h.size();
  std::vector<int64_t> order(m);
  std::iota(order.begin(), order.end(), 0);
  std::sort(order.begin(), order.end(), [&](int64_t x, int64_t y) {
    return keys[2 * x] != keys[2 * y] ? keys[2 * x] < keys[2 * y] : keys[2 * x + 1] < keys[2 * y + 1];
  });
  *n_out = m;
  for (int64_t k = 0; k < m && k < cap; ++k) {
    keys_out[2 * k] = keys[2 * order[k]]; keys_out[2 * k + 1] = keys[2 * order[k] + 1]; h_out[k] = h[order[k]];
  }
  return m > cap ? DH_EINVAL : DH_OK;
}

dh_status detham_diagonals(detham_ctx* c, const uint64_t* dets, int64_t m, double* out) {
  if (!c || !dets || !out || m < 0) return DH_EINVAL;
  if (m == 0) return DH_OK;
  dh_status st = dh_diagonals(c, reinterpret_cast<const u64*>(dets), m, out);
  if (st != DH_OK) return st;
  DH_CUDA(c, cudaStreamSynchronize(c->stream));
  return DH_OK;
}

dh_status detham_get_counters(detham_ctx* c, detham_counters* out) {
  if (!c || !out) return DH_EINVAL;
  *out = c->ctr;
  return DH_OK;
}

void detham_destroy(detham_ctx* c) {
  if (!c) return;
  cudaStreamSynchronize(c->stream);
  free_all(c);
  delete c;
}

const char* detham_strerror(dh_status s) {
  switch (s) {
    case DH_OK: return "ok";
    case DH_EINVAL: return "invalid argument";
    case DH_EUNSORTED: return "subspace not strictly ascending (unsorted or duplicate determinants)";
    case DH_EPOPCOUNT: return "determinant with wrong electron count or orbital index out of range";
    case DH_ENOMEM: return "out of memory";
    case DH_ETABLEFULL: return "PT2 hash table full (raise table_slots or n_parts)";
    case DH_ECUDA: return "CUDA error";
  }
  return "unknown status";
}

const char* detham_last_cuda_error(detham_ctx* c) { return c ? c->cuda_err.c_str() : ""; }

}  // extern "C"
