/* detham.h — C ABI of the B200-native combinatorial Hamiltonian kernel of arxiv 2601.21310.
 *
 * The library rebuilds on one GPU (sm_100a) the paper's "Discrete Combinatorial Kernel" (Layer 0:
 * "Evaluates Slater-Condon rules on integer representations of configurations to construct the Hamiltonian
 * connectivity graphs (H_VV, H_VP) ... exporting sparse operators in CSR format"), the host-resident SpMV
 * v = H psi (Alg. 1 line 14 at PAPER.md:282), the variational energy E_var (Eq. 11) and
 * the external Epstein-Nesbet PT2 term (Eq. 13 second term) with heat-bath screening
 * (Eq. 14 and the tau rule).  The paper calls the variational set V; here it is S.
 *
 * Conventions
 *  - Plain C, no exceptions cross the boundary; every call returns a dh_status.
 *  - n_orb = number of SPATIAL orbitals, 1 <= n_orb <= 64.  A determinant is two uint64 words {alpha, beta}; bit p of a
 *    word = spatial orbital p occupied in that spin string.  |D> = prod_{p in alpha, ascending} a+_{p alpha}
 *    prod_{q in beta, ascending} a+_{q beta} |0>  (sign convention; reading Q1).
 *  - Integrals: h1 fp64 [n_orb*n_orb] symmetric; eri fp64 packed 8-fold symmetric chemist-notation (pq|rs) at
 *    eri[T(T(p,q), T(r,s))], T(x,y) = max(x,y)*(max(x,y)+1)/2 + min(x,y)  (reading Q3).
 *  - "device" pointers are CUDA device memory on the current device; "host" pointers are ordinary host memory.
 *    Inputs are BORROWED (the caller keeps ownership; `dets` must stay valid until the next detham_set_subspace or
 *    detham_destroy).  Everything reachable through detham_csr is OWNED by the context.
 *  - All work is enqueued on the stream given at creation; calls that return scalars to host memory synchronise that
 *    stream before returning.
 *  - Nothing is truncated or sorted silently: an unsorted S, a full hash table or an allocation failure is an error code.
 *  - There is no CPU fallback: without a CUDA device every compute call returns DH_ECUDA.
 */
#ifndef DETHAM_H
#define DETHAM_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct detham_ctx detham_ctx; /* opaque; owns every device allocation it makes */

typedef enum {
  DH_OK = 0,
  DH_EINVAL = 1,     /* bad argument (NULL, n_orb out of range, negative or NaN threshold, call order) */
  DH_EUNSORTED = 2,  /* S not strictly ascending by (alpha, beta) (covers duplicates) */
  DH_EPOPCOUNT = 3,  /* a determinant has the wrong electron count or a bit at or above n_orb */
  DH_ENOMEM = 4,     /* device or host allocation failed */
  DH_ETABLEFULL = 5, /* PT2 hash table overflowed with the configured capacity / partition count */
  DH_ECUDA = 6       /* CUDA runtime error (no device, launch failure); see detham_last_cuda_error */
} dh_status;

/* Counters of the most recent calls (metrics). */
typedef struct {
  int64_t nnz;              /* stored entries of H_SS (diagonal included) */
  int64_t build_generated;  /* candidates ham_build looked up in S: the doubles that passed the screen and every single (singles are
                               looked up first and evaluated only when they are in S) */
  int64_t pt2_generated;    /* excitations that passed the screen in pt2 (members of S included) */
  int64_t pt2_contrib;      /* contributions H_ai psi_i added to externals a not in S */
  int64_t pt2_external;     /* distinct externals */
  int32_t pt2_parts;        /* key partitions (passes) used by the last pt2 */
  int32_t pt2_max_probe;    /* longest probe sequence seen */
  int64_t pt2_table_slots;  /* slots of the hash table used by each pass */
  int64_t pt2_probe_parts;  /* 0, or the partition count of the one-slice probe the planner ran to measure duplication */
  double pt2_sum_abs;       /* sum_a |v_a^2 / (E_S - H_aa)| / psi^T psi  (conditioning report, reading Q11) */
  double pt2_min_abs_den;   /* min_a |E_S - H_aa| */
  /* device times (CUDA events on the context's stream) of the kernels of the last calls, milliseconds */
  double ms_store;          /* set_subspace: validation + lookup-index build */
  double ms_build_count;    /* ham_build enumeration pass (enumerate + lookup, hits appended to an arena) + row scan;
                               includes the exact-size rerun when the arena of the previous build was too small */
  double ms_build_fill;     /* ham_build arena -> CSR copy + per-row column sort */
  double ms_energy;         /* SpMV + fused reductions */
  double ms_pt2_plan;       /* pt2 class histogram (pass planning), 0 when both table_slots and n_parts are configured */
  double ms_pt2_accum;      /* pt2 member insert + enumerate/accumulate kernels, summed over passes */
  double ms_pt2_scan;       /* pt2 table scan/clear + reductions, summed over passes */
  int64_t hsp_nnz;          /* stored entries of H_SP (last detham_hsp_build) */
  int64_t hsp_generated;    /* excitations that passed the screen in hsp_build (looked up in P) */
  double ms_hsp_build;      /* hsp_build enumeration pass (enumerate + lookup in P, hits appended to the arena) + row scan */
  double ms_hsp_fill;       /* hsp_build arena -> CSR copy + per-row column sort */
  int64_t pt2_binned;       /* organisation of the last pt2: 0 = hash table in HBM probed directly, 1 = hash table in HBM with binned
                               passes, 2 = streamed (records partitioned by key region, deduplicated in L2-resident region tables;
                               no table in HBM) */
  int64_t pt2_stream_bins;  /* streamed organisation: key regions per pass (0 otherwise); pt2_table_slots = slots of one region table */
  int64_t build_pairs;      /* 1 if the last ham_build went by excitation degree (pairs of S), 0 if it walked the heat-bath lists;
                               build_generated then counts the Slater-Condon elements evaluated */
} detham_counters;

/* Options of pt2 (SURVEY.md section 5 "config / flag system").  Zero in every field = the defaults. */
typedef struct {
  int32_t mode;             /* 0 = choose (today: the hash table in HBM, with binned passes when it is far beyond L2);
                               1 = hash table in HBM; 2 = streamed (DH_EINVAL if |S| < 16 x SM count) */
  int32_t n_parts;          /* key partitions / passes, a power of two <= 1024 (streamed: <= 256); 0 = planned */
  int64_t table_slots;      /* table organisation: capacity in 32-byte slots; 0 = planned from free device memory */
  double table_load;        /* table organisation: target load factor; 0 = 0.5, and 0.6 for binned passes of large tables (their
                               probes are L2 hits, a denser table is less DRAM traffic: measured) */
  double max_table_gb;      /* table organisation: the planner never sizes the table beyond this (random 32-byte accesses lose
                               4x of their rate past ~70 GB on a B200: TLB reach); 0 = 60 */
  double small_den;         /* externals with |E_S - H_aa| below this take H_aa from the key alone instead of the O(1) update from
                               the source that claimed them (its rounding, ~1e-13, is amplified by 1 / denominator; DESIGN.md
                               reading Q11); 0 = 1e-3, negative = never */
  int32_t stream_bins;      /* streamed: key regions per pass (<= 4096); 0 = planned so that a region's distinct keys fit its table */
  int32_t table_regions;    /* table organisation, binned passes (contributions appended per table region, then merged region by
                               region so that the probes stay in L2): 0 = when the table exceeds 8 GB (and the record pool fits), with at most 2048 regions;
                               > 0 = always, with at most that many regions (64..8192); -1 = never */
  double stream_ring_mb;    /* streamed: bytes of the three region tables together (they must stay in L2); 0 = 96 */
  double stream_load;       /* streamed: target load factor of a region table; 0 = 0.45 */
  double stream_pool_frac;  /* head room of the record pool over the planned estimate (streamed: 0 = 1.15; binned passes: 0 = 1.2) */
  double stream_pool_gb;    /* streamed: budget of the record pool; 0 = 80 % of the free device memory */
} detham_pt2_options;

/* Create a context: uploads the integrals, derives J_pq = (pp|qq), K_pq = (pq|qp), and builds the heat-bath lists
 * ("we precompute a lookup table during initialization: for each pair of occupied spin-orbitals (i,j),
 * the corresponding pairs of virtual orbitals (a,b) are sorted in descending order of the integral magnitude").
 * h1 / eri: host OR device pointers (detected).  cuda_stream: a cudaStream_t cast to void*, NULL = default stream.
 * Requires 1 <= n_orb <= 64, 0 <= n_alpha, n_beta <= n_orb, n_alpha + n_beta >= 1. */
dh_status detham_create(detham_ctx** out, int n_orb, int n_alpha, int n_beta, const double* h1, const double* eri,
                        double e_core, void* cuda_stream);

/* Set the variational subspace S ("variational set V_k").  dets: DEVICE uint64 [n_dets][2] = {alpha, beta},
 * strictly ascending as 128-bit numbers with alpha the high word; 1 <= n_dets < 2^31.  Validated on the device
 * (DH_EUNSORTED / DH_EPOPCOUNT).  Builds the L2-resident lookup structure of the determinant store.  Invalidates any CSR. */
dh_status detham_set_subspace(detham_ctx* ctx, const uint64_t* dets, int64_t n_dets);

/* ham_build (Alg. 1 line 8: "Construct sparse Hamiltonian block H_VV"): CSR with row i =
 * {(i, H_ii)} U {(j, H_ij) : D_j in S, D_j a single or double excitation of D_i, |H_ij| >= eps, H_ij != 0}, columns
 * ascending (reading Q4).  eps >= 0.  *nnz_out (host, may be NULL) receives the number of stored entries. */
dh_status detham_ham_build(detham_ctx* ctx, double eps, int64_t* nnz_out);

/* Choose how ham_build finds the connections inside S: 0 = the library chooses; 1 = walk the heat-bath lists of every source and
 * look the screened excitations up in S; 2 = by excitation degree: pairs of S whose bit strings differ by at most
 * a double excitation (|S| <= 2^31).  Both give the same CSR, bit for bit off the diagonal. */
dh_status detham_build_config(detham_ctx* ctx, int method);

/* Device pointers of the CSR built last: row_ptr int64 [n_dets+1], col int32 [nnz], val fp64 [nnz].  Valid until the next
 * detham_ham_build / detham_set_subspace / detham_destroy.  DH_EINVAL if no CSR exists. */
dh_status detham_csr(detham_ctx* ctx, const int64_t** row_ptr, const int32_t** col, const double** val);

/* Copy the CSR built last into caller buffers (each HOST or DEVICE, detected; any may be NULL to skip):
 * row_ptr int64 [n_dets+1], col int32 [nnz], val fp64 [nnz].  Synchronises the stream. */
dh_status detham_csr_copy(detham_ctx* ctx, int64_t* row_ptr, int32_t* col, double* val);

/* energy (Eq. 11; the SpMV of Alg. 1 line 14): y = H_SS psi, E_S = psi^T y / psi^T psi.
 * psi: DEVICE fp64 [n_dets].  y_out: DEVICE fp64 [n_dets] or NULL.  e_out, norm2_out: HOST (norm2_out may be NULL).
 * DH_EINVAL if psi^T psi is zero or not finite (y_out is written all the same). */
dh_status detham_energy(detham_ctx* ctx, const double* psi, double* e_out, double* norm2_out, double* y_out);

/* energy for callers that may not allocate (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc):
 * the same per-row arithmetic as detham_energy (Eq. 11) on a CSR the caller passes, with the partial sums in a
 * file-scope device array of the library (128 KB, held by every GPU that loads the library until exit) instead of a buffer of
 * a context.  The call needs no context, allocates nothing (no cudaMalloc, cudaFree or allocating library routine), does not
 * synchronise, and launches two kernels on `stream` (a cudaStream_t; NULL = the default stream) of the CURRENT device.
 *   row_ptr DEVICE int64 [n_dets+1], col DEVICE int32 [nnz], val DEVICE fp64 [nnz], psi DEVICE fp64 [n_dets]: borrowed inputs,
 *     e.g. from detham_csr; n_dets >= 1; nnz (the number of stored entries) only chooses the threads per row.
 *   y_out DEVICE fp64 [n_dets] or NULL: y = H psi.
 *   out3 DEVICE fp64 [3]: {psi^T H psi, psi^T psi, E_S = their quotient}, written on `stream`.
 * Sums are taken per block of 1024 rows and then over the blocks in a fixed order: the result is reproducible and does not
 * depend on the GPU, but differs from detham_energy's in the last bits (another order of the same additions).
 * Errors: DH_EINVAL for a NULL pointer, n_dets < 1, or n_dets > DETHAM_ENERGY_STATIC_MAX_ROWS (nothing is launched);
 * DH_ECUDA for a CUDA failure; detham_energy_static_error() gives the text for the calling thread ("" after a success).
 * Every call on a device shares the one array, which keeps the last call's contents: each entry read is written first by the
 * same call, so nothing is cleared, but calls that OVERLAP on the GPU (different streams, or replays of captured graphs in
 * flight together) race on it - run them in stream order. */
#define DETHAM_ENERGY_STATIC_MAX_ROWS 8388608 /* 2^23 determinants */
dh_status detham_energy_static(const int64_t* row_ptr, const int32_t* col, const double* val, const double* psi,
                               int64_t n_dets, int64_t nnz, double* y_out, double* out3, void* stream);
const char* detham_energy_static_error(void);

/* residual: r = H_SS psi - e_s psi, the vector that Eq. 12 contracts with grad psi,
 * and the internal term of Eq. 13 (first sum) on the CSR built last (reading Q4: the screened
 * operator): *internal_out = (1 / psi^T psi) sum_{i in S} r_i^2 / (e_s - H_ii); a row with r_i == 0 contributes 0.
 * psi: DEVICE fp64 [n_dets]; r_out: DEVICE fp64 [n_dets] or NULL; internal_out: HOST.  No regularisation of the denominators. */
dh_status detham_residual(detham_ctx* ctx, const double* psi, double e_s, double* r_out, double* internal_out);

/* ediag: E_diag = lambda_min(H_SS) of the CSR built last, by Lanczos on the device
 * (SpMV = the energy kernel).  v0: DEVICE fp64 [n_dets] start vector (psi is a good one) or NULL (all ones).  With r the residual
 * norm ||H y - theta y|| of the smallest Ritz pair (an eigenvalue lies within r of theta), the iteration stops when
 * r <= tol |theta| or when the Krylov space closes; otherwise after max_iter steps with *converged_out = 0 (the value is then an
 * upper bound of lambda_min only).  theta itself converges like r^2 / gap, so tol = 1e-8 already gives ~1e-12 on the value.
 * e_out, iters_out, resid_out (= r), converged_out (1 / 0): HOST, all but e_out may be NULL.  Delta_opt of the paper =
 * E_S - *e_out >= 0. */
dh_status detham_ediag(detham_ctx* ctx, const double* v0, double tol, int max_iter, double* e_out, int* iters_out,
                       double* resid_out, int* converged_out);

/* Configure pt2: table_slots = hash-table capacity in 32-byte slots (0 = choose from free device memory);
 * n_parts = number of key partitions / passes, a power of two <= 1024 (0 = choose so that every partition fits).
 * Shorthand for the two fields of the same name of detham_pt2_options; the other options keep their values. */
dh_status detham_pt2_config(detham_ctx* ctx, int64_t table_slots, int n_parts);

/* Set every option of pt2 (opts == NULL: back to the defaults).  DH_EINVAL for values out of range; nothing is changed then. */
dh_status detham_pt2_set_options(detham_ctx* ctx, const detham_pt2_options* opts);

/* Release the large work buffers of pt2 (hash table, record pool, region tables, cached heat-bath list splits other than the
 * unsplit one); they are re-created on demand.  For callers that share the device with other allocations. */
dh_status detham_trim(detham_ctx* ctx);

/* pt2 (Eq. 13 second term, screened per Eq. 14 / PAPER.md:227; readings Q6, Q9, Q10):
 * for every source i with psi_i != 0, tau_i = eps2 / |psi_i| (0 if eps2 == 0); for every single or double excitation a
 * of D_i with |H_ai| >= tau_i, H_ai != 0 and a not in S:  v_a += H_ai psi_i.
 * Result  dE = (1 / psi^T psi) sum_a v_a^2 / (e_s - H_aa).  psi: DEVICE fp64 [n_dets]; outputs HOST (counts may be NULL).
 * DH_EINVAL if psi^T psi is zero or not finite. */
dh_status detham_pt2(detham_ctx* ctx, const double* psi, double e_s, double eps2, double* pt2_out,
                     int64_t* n_external_out, int64_t* n_contrib_out);

/* Size of the screened connected set (Eq. 1 with the screen of Eq. 14), summed over the sources:
 *   psi == NULL: sum_i |{ x' : x' a single or double excitation of D_i, |H_x'i| >= thr, H != 0 }|   (the screen of ham_build)
 *   psi != NULL (DEVICE fp64 [n_dets]): the same with tau_i = thr / |psi_i|, rows with psi_i == 0 skipped (the screen of pt2).
 * Members of S and externals alike; every single is evaluated.  A property of the input, independent of how ham_build and pt2
 * are organised: the benchmark's "Hamiltonian elements" are count(NULL, eps) + count(psi, eps2).  *n_out: HOST. */
dh_status detham_count_screened(detham_ctx* ctx, const double* psi, double thr, int64_t* n_out);

/* expand (Alg. 1 "Subspace Expansion"): the perturbative set of Eq. 14
 *   P = { a not in S : max_i |H_ai psi_i| >= eps2 },
 * generated by the same screened enumeration as pt2 (an external belongs to P iff it is generated at least once), written
 * deduplicated and sorted ascending by (alpha, beta) with, per external: score = max_i |H_ai psi_i|, v = sum_i H_ai psi_i over the
 * generated couplings (reading Q9) and H_aa (from scratch).  All buffers DEVICE: keys_out uint64 [cap][2]; score_out, v_out,
 * haa_out fp64 [cap], each may be NULL.  *n_out (HOST) = |P|; if |P| > cap nothing is written and the call returns DH_EINVAL
 * with *n_out set, so a first call with cap = 0 sizes the buffers.  |P| < 2^32. */
dh_status detham_expand(detham_ctx* ctx, const double* psi, double eps2, uint64_t* keys_out, double* score_out, double* v_out,
                        double* haa_out, int64_t cap, int64_t* n_out);

/* hsp_build ("constructs the sparse Hamiltonian blocks H_VV and H_VP in CSR format"; H_VP
 * of Eq. S3; the V-P block of the Proxy Hamiltonian, Eq. 8): CSR with one row per determinant of S
 * and one column per entry of `pkeys` - DEVICE uint64 [m][2], strictly ascending by (alpha, beta), same electron counts as S
 * (DH_EUNSORTED / DH_EPOPCOUNT otherwise): the output of detham_expand or any sorted subset a selector kept; borrowed for the
 * duration of the call only.  Row i holds H_{P_k, i} for every coupling the screen of Eq. 14 generates from source i
 * (|H| >= eps2 / |psi_i|, H != 0; rows with psi_i == 0 are empty: readings Q6, Q9) whose target is in `pkeys`; columns ascending.
 * The P-P block of Eq. 8 is diagonal: it is detham_expand's haa_out (or detham_diagonals).  psi: DEVICE fp64 [n_dets].
 * m < 2^31, may be 0.  *nnz_out (HOST, may be NULL).  The CSR is owned by the context (detham_hsp_csr / detham_hsp_csr_copy),
 * valid until the next detham_hsp_build / detham_set_subspace / detham_destroy. */
dh_status detham_hsp_build(detham_ctx* ctx, const double* psi, double eps2, const uint64_t* pkeys, int64_t m, int64_t* nnz_out);

/* complete_sum (the complete-the-sum variant; Eq. 13, PAPER.md:189 writes the external numerator as
 * <x|H|Psi_V>, the full projection, while Eq. 14 / PAPER.md:227 generate only the couplings above the screen - DESIGN.md reading
 * Q9): for `pkeys` - DEVICE uint64 [m][2], strictly ascending, same electron counts as S (DH_EUNSORTED / DH_EPOPCOUNT otherwise),
 * normally the keys detham_expand selected - v_out[k] = sum over ALL i in S of H_{P_k, i} psi_i, screened or not (a key that is
 * itself a member of S includes its diagonal term).  One unscreened enumeration of every source with psi_i != 0, so the cost is
 * that of pt2 at eps2 = 0.  psi: DEVICE fp64 [n_dets]; v_out: DEVICE fp64 [m], overwritten; m < 2^31, may be 0.  The additions
 * are atomic: their order, hence the last bits, vary from run to run.  Synchronises the stream. */
dh_status detham_complete_sum(detham_ctx* ctx, const double* psi, const uint64_t* pkeys, int64_t m, double* v_out);
/* Device pointers of H_SP: row_ptr int64 [n_dets+1], col int32 [nnz], val fp64 [nnz].  DH_EINVAL if none exists. */
dh_status detham_hsp_csr(detham_ctx* ctx, const int64_t** row_ptr, const int32_t** col, const double** val);
/* Copy H_SP into caller buffers (each HOST or DEVICE, detected; any may be NULL to skip).  Synchronises the stream. */
dh_status detham_hsp_csr_copy(detham_ctx* ctx, int64_t* row_ptr, int32_t* col, double* val);

/* Per-partition partial sums (already divided by psi^T psi) of the last detham_pt2; writes min(cap, n_parts) values to
 * `out` (HOST) and the partition count to *n_parts_out. */
dh_status detham_pt2_partials(detham_ctx* ctx, double* out, int cap, int* n_parts_out);

/* Whole hot path from HOST buffers (the end-to-end entry): copies dets and psi to the device, then set_subspace ->
 * ham_build(eps) -> energy -> pt2(E_S, eps2), and returns the scalars to host memory. */
dh_status detham_solve_host(detham_ctx* ctx, const uint64_t* dets_host, const double* psi_host, int64_t n_dets,
                            double eps, double eps2, double* e_out, double* pt2_out, int64_t* nnz_out,
                            int64_t* n_external_out);

/* Test hook: the full screened connection list of source `row` of S at cutoff tau (members of S and externals alike,
 * diagonal excluded), sorted by key.  keys_out HOST uint64 [cap][2], h_out HOST fp64 [cap]; *n_out = number found
 * (if > cap only cap entries are written and the call returns DH_EINVAL). */
dh_status detham_connections(detham_ctx* ctx, int64_t row, double tau, uint64_t* keys_out, double* h_out, int64_t cap,
                             int64_t* n_out);

/* Test hook: H_aa for `m` arbitrary determinants (DEVICE uint64 [m][2]) into DEVICE fp64 [m]. */
dh_status detham_diagonals(detham_ctx* ctx, const uint64_t* dets, int64_t m, double* out);

dh_status detham_get_counters(detham_ctx* ctx, detham_counters* out);
void detham_destroy(detham_ctx* ctx);
const char* detham_strerror(dh_status s);
const char* detham_last_cuda_error(detham_ctx* ctx); /* text of the last CUDA error seen by this context, "" if none */

#ifdef __cplusplus
}
#endif
#endif /* DETHAM_H */
