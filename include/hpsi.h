/*
 * hpsi.h - C ABI of the B200-native effective-Hamiltonian application for two-site QC-DMRG.
 *
 * What is computed (BASELINE.json `north_star`; "Numerical procedure" names the step:
 * "solving a large hermitian eigenvalue problem using e.g. the Lanczos or Davidson method. This step
 * usually accounts for 80% of the execution time, and scales as O(D^3)"):
 *
 *     psi'(l,r) = sum_t  c_t * A_t(l,l') * psi(l',r') * B_t(r,r')^T
 *
 * in block-sparse symmetry-sector form, real FP64 (Fig. 1 "FP64"), plain transpose.
 * Index convention (reading A2):  out[x,y] = sum_{x',y'} A[x,x'] * psi[x',y'] * B[y,y'].
 *
 * Layout of psi / out: for left sector i = 0..n_left-1
 * ascending, if a right sector j with q_left[i] + q_right[j] == target exists, psi holds the dense
 * d_left[i] x d_right[j] block, row-major, appended to the vector.  hpsi_query(HPSI_Q_PSI_BLOCKS) returns it.
 *
 * Pointers: every argument says HOST or DEVICE.  No C++ exception crosses this boundary; every call
 * returns 0 on success or a negative HPSI_E* code, and hpsi_last_error() gives a thread-local message.
 * The library has no CPU fallback: without a CUDA device every compute entry point fails with HPSI_ECUDA.
 */
#ifndef HPSI_H_
#define HPSI_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define HPSI_OK       0
#define HPSI_EINVAL  (-1)   /* malformed sector table / term list / argument                         */
#define HPSI_ENOMEM  (-2)   /* host or device allocation failed                                      */
#define HPSI_ECUDA   (-3)   /* CUDA runtime error (message holds cudaGetErrorString)                 */
#define HPSI_ESTATE  (-4)   /* call not valid in the plan's state (arenas not bound, host-only plan) */

/* hpsi_plan flags */
#define HPSI_PLAN_HOST_ONLY  (1u << 0)  /* build the schedule on the host only: no CUDA call, no device memory.
                                           Such a plan serves hpsi_query and hpsi_debug_* ; hpsi_apply -> ESTATE. */
#define HPSI_PLAN_FIXED_ORDER1 (1u << 1) /* diagnostic: force (A psi) B^T for every task                  */
#define HPSI_PLAN_FIXED_ORDER2 (1u << 2) /* diagnostic: force A (psi B^T) for every task                  */
#define HPSI_PLAN_NO_FUSION    (1u << 3) /* every task goes through the two-launch path with the workspace (the default)  */
#define HPSI_PLAN_FUSE_ALL     (1u << 4) /* run every task that fits one CTA tile through the fused kernel: both GEMMs in
                                            one CTA, the intermediate kept in shared memory        */

typedef struct hpsi_plan hpsi_plan_t;   /* opaque; owns the device schedule and the workspace */

/* "Sector table" (north_star).  All arrays HOST, copied by hpsi_plan. */
typedef struct {
  int32_t n_left, n_right;
  const int32_t* q_left;    /* [n_left][2]  labels (N, 2Sz); unique within the side (else EINVAL) */
  const int32_t* q_right;   /* [n_right][2]                                                      */
  const int32_t* d_left;    /* [n_left]  sector dimensions, each >= 1                            */
  const int32_t* d_right;   /* [n_right]                                                         */
  int32_t target[2];        /* Q* = (N*, 2Sz*)                                                   */
} hpsi_sectors_t;

/* One dense operator block: maps sector `col` to sector `row` of its side; rows x cols = d[row] x d[col],
 * row-major with leading dimension ld >= d[col], starting `offset` doubles into the side's arena. */
typedef struct {
  int32_t term, row, col, ld;
  int64_t offset;
} hpsi_opblock_t;

/* "Term list" (north_star).  Descriptors and coef are HOST (copied).  a_data / b_data are DEVICE arenas,
 * caller-owned and BORROWED: they must outlive the plan (no copy is made - at D=8192 they are ~80 GB).
 * They may be NULL at plan time and bound later with hpsi_bind.  a_len / b_len = arena lengths in doubles
 * (used to validate descriptors).  Fast path (TMA staging): every block has even `offset` and even `ld` and the
 * arenas are 16-byte aligned; preferred: `ld` and `offset` multiples of 4 (rows start on a 32-byte L2 sector).
 * Anything else runs an 8-byte cp.async variant of the kernels (correct, slower).  Padding elements are never
 * read into a result (out-of-range rows / columns are zero-filled on the way into shared memory). */
typedef struct {
  int32_t n_terms;
  const double* coef;              /* [n_terms] c_t                                             */
  int64_t n_a;
  const hpsi_opblock_t* a_blocks;  /* [n_a] any order; at most one block per (term,row,col)       */
  int64_t n_b;
  const hpsi_opblock_t* b_blocks;  /* [n_b]                                                      */
  const double* a_data;            /* DEVICE (or NULL)                                           */
  const double* b_data;            /* DEVICE (or NULL)                                           */
  int64_t a_len, b_len;
  /* Adjoint-pair storage sharing: HOST, [n_a] / [n_b], may be NULL (= all zero).  A non-zero entry
   * says the arena holds the TRANSPOSE of that block: element (x, x') of the block is arena[offset + x' * ld + x] with
   * ld >= d[row].  A Hermitian H pairs every term with its adjoint (same c, A^T, B^T): the adjoint term's descriptors
   * can then point at the base term's storage and the operator arenas halve (80 -> 40 GB at D=8192).  Such blocks are
   * staged K-major (TMA boxes of 8 rows x 16 k, 64-byte swizzle); tiles stay padded to 8 rows as in plain plans.
   * The flags are per block and independent: any mix of plain and transposed A / B blocks inside a term is legal. */
  const uint8_t* a_transposed;
  const uint8_t* b_transposed;
} hpsi_terms_t;

/* Steps 1-4 of SURVEY.md 8(a): psi block table, task enumeration, per-task order choice
 * (A psi)B^T vs A(psi B^T) by flop count, grouping of all tasks that write one output block, cutting into
 * CTA work units; uploads the flat schedule and allocates the workspace.  One-off, synchronous. */
int hpsi_plan(const hpsi_sectors_t* sectors, const hpsi_terms_t* terms, uint32_t flags, hpsi_plan_t** plan_out);

/* hpsi_plan with options.  options == NULL is hpsi_plan.
 *   struct_bytes        sizeof(hpsi_plan_options_t) as the caller compiled it (lets the struct grow)
 *   shard_of_term       HOST int32[n_terms] or NULL.  Term sharding for the multi-GPU apply (PAPER.md:27
 *                       "hybrid CPU-multi GPU", "eight GPU accelerated diagonalization procedure"): only the
 *                       terms with shard_of_term[t] == shard_index are planned.  The blocks of every other term are
 *                       ignored and not validated, so the arenas need hold the shard's blocks only (operators are the
 *                       13-80 GB object; psi is replicated).  The sum over shard_index of the shards' H psi is H psi.
 *                       hpsi_shard_terms below produces a balanced assignment.
 *   p1_stages_per_unit  schedule knobs, 0 = automatic: staged K-tiles per CTA of the first-GEMM kernel; waves of CTAs the
 *   p2_waves            second GEMM's split-K aims at; least DMMA count per second-GEMM CTA.  They change the schedule
 *   p2_min_unit_dmma    (and so the rounding order of the sums), never the result beyond that; HPSI_Q_TUNING reports
 *                       the values a plan was built with.
 *   n_vectors           k > 1 plans a BATCHED apply (hpsi_apply_multi): the k vectors widen the first GEMM's N dimension
 *                       and multiply the second GEMM's tiles, so the operators stream from HBM once for k products - what a
 *                       block (multi-root) Davidson calls.  Workspace grows k-fold.  Not available for plans
 *                       with transposed blocks or HPSI_PLAN_FUSE_ALL (EINVAL).  Queries of flops / bytes stay per vector. */
typedef struct {
  uint32_t struct_bytes;
  int32_t shard_index;
  const int32_t* shard_of_term;
  int32_t p1_stages_per_unit;
  int32_t p2_waves;
  int32_t p2_min_unit_dmma;
  int32_t n_vectors;              /* 0 or 1: single-vector plan; k > 1: lay the plan out for hpsi_apply_multi on up to k vectors */
} hpsi_plan_options_t;
int hpsi_plan_ex(const hpsi_sectors_t* sectors, const hpsi_terms_t* terms, uint32_t flags,
                 const hpsi_plan_options_t* options, hpsi_plan_t** plan_out);

/* Balanced partition of the term list over `shard_count` ranks ("Partition the terms (balanced by
 * useful_flops ...)").  HOST only, deterministic (every rank computes the same answer): bundles of terms are sorted by
 * useful flops (descending, ties by lowest term) and dealt greedily to the lightest shard so far (ties: lowest index).
 *   terms              descriptors only (coef, arenas, ld and offset are not read)
 *   bundle_of_term     HOST int32[n_terms] or NULL: terms with the same value stay on one rank - e.g. a term and its
 *                      adjoint when the adjoint reads its partner's storage (a_transposed); NULL = every term alone
 *   shard_of_term      HOST out, int32[n_terms], values 0..shard_count-1
 *   shard_flops        HOST out or NULL, int64[shard_count]: useful flops of every shard */
int hpsi_shard_terms(const hpsi_sectors_t* sectors, const hpsi_terms_t* terms, const int32_t* bundle_of_term,
                     int32_t shard_count, int32_t* shard_of_term, int64_t* shard_flops);

/* The operator-arena layout the kernels like best, written into the descriptors (SURVEY.md 8(b) "preferred ld / arena
 * layout"; HPSI_Q_PREFERRED_LAYOUT gives the rule as numbers).  For every descriptor, in the order given: ld = stored
 * columns rounded up to 4 doubles, offset = running total rounded up to 4 doubles (every row starts on a 32-byte L2
 * sector and is a legal TMA row).  A block flagged transposed stores d[col] x d[row].  Blocks with ld == -1 on input
 * share storage with another descriptor and are skipped (the caller copies offset / ld from its partner).
 * blocks: HOST, in/out; d: HOST sector dims of that side; transposed: HOST or NULL; arena_len: HOST out, doubles.
 * Use: describe -> hpsi_layout_blocks (both sides) -> fill the arenas -> hpsi_plan (arenas may be NULL) -> hpsi_bind. */
int hpsi_layout_blocks(int32_t n_sectors, const int32_t* d, int64_t n_blocks, hpsi_opblock_t* blocks,
                       const uint8_t* transposed, int64_t* arena_len);

/* (Re)bind the DEVICE operator arenas (same descriptors).  Re-encodes the tensor maps of the operand matrices
 * (host work proportional to the number of blocks; synchronous). */
int hpsi_bind(hpsi_plan_t* plan, const double* a_data_dev, const double* b_data_dev);

/* Per-task coupling coefficients (reading A4): replaces the coefficient of every task,
 * which hpsi_plan initialises to c_term - e.g. SU(2) recoupling factors that depend on the sector quadruple
 * (l, l', r, r') and not only on the term ("spin adapted", "SU(2)-aware").
 * coef_host: HOST, n doubles with n == HPSI_Q_N_TASKS, in HPSI_Q_TASKS order (copied before the call returns).
 * Stream-ordered: the device tables are updated by copies enqueued on cuda_stream, so applies enqueued on that stream
 * before the call see the old values and applies enqueued after it the new ones; no device-wide synchronisation.
 * hpsi_apply, hpsi_diagonal, hpsi_davidson and hpsi_lanczos all use the new values. */
int hpsi_set_task_coefficients(hpsi_plan_t* plan, const double* coef_host, int64_t n, void* cuda_stream);

/* Steps 5-7: out = H psi (overwrite).  psi_dev / out_dev: DEVICE, psi_length doubles each, must not alias.
 * cuda_stream: a cudaStream_t cast to void* (NULL = default stream).  Enqueue only: no host sync, no
 * allocation, CUDA-graph capturable.  A plan owns one workspace: do not run it on two streams at once.
 * Repeated applies on the same inputs are bitwise identical (no atomics on data).
 * Launch form (all entry points): every kernel is enqueued as a programmatic dependent of the operation before it in
 * the stream and waits on the device (griddepcontrol.wait) before its first memory access, which hides its launch latency
 * (~2 us per kernel boundary).  Stream order and visibility are those of plain launches: the caller's own work before
 * and after a call needs no change. */
int hpsi_apply(hpsi_plan_t* plan, const double* psi_dev, double* out_dev, void* cuda_stream);

/* Batched apply: out_v = H psi_v for v = 0 .. n_vectors-1 in one pass over the operators (plan built with
 * hpsi_plan_options_t.n_vectors >= n_vectors).  Vector v of psi starts at psi_dev + v * ld_psi, of out at out_dev + v * ld_out
 * (ld_* >= psi_length; the two sets must not overlap).  Same kernels, same launches as hpsi_apply; every vector's result
 * is bitwise what hpsi_apply_multi gives for it in any batch of the same plan.  Enqueue only, CUDA-graph capturable. */
int hpsi_apply_multi(hpsi_plan_t* plan, const double* psi_dev, int64_t ld_psi, double* out_dev, int64_t ld_out,
                     int32_t n_vectors, void* cuda_stream);

/* Exchange step of the term-sharded apply: out[i] = parts[0*n + i] + parts[1*n + i] + ... added in
 * that order.  Each rank hpsi_apply's its shard, the partial results are all-gathered (NCCL; psi' is 5-17 MB) into
 * parts_dev in rank order, and this sum gives every rank the same bits on every run - a library all-reduce does not
 * promise its summation order.  parts_dev: DEVICE, n_parts * n doubles; out_dev: DEVICE, n doubles, may equal
 * parts_dev (in place over shard 0) but must not overlap it otherwise.  Enqueue only. */
int hpsi_sum_shards(const double* parts_dev, int32_t n_parts, int64_t n, double* out_dev, void* cuda_stream);

/* Eigensolvers on a term-sharded plan ("eight GPU accelerated diagonalization procedure"):
 * every rank runs the same hpsi_davidson / hpsi_davidson_multi / hpsi_lanczos call on its shard plan with the same start
 * vector, and the solver hands every product it computes to `fn` before using it:
 *   fn(user, v_dev, w_dev, n, n_vectors, ld, cuda_stream)
 *     w_dev   DEVICE, in/out: n_vectors vectors of n doubles, ld doubles apart - on entry this rank's partial results
 *             (the sum over ITS terms), on return (stream order) the sum over all ranks
 *     v_dev   DEVICE, the vectors that were multiplied (same layout), or NULL when w_dev is the partial diag(H)
 *   fn only enqueues on cuda_stream (e.g. NCCL all-gather of w + hpsi_sum_shards in rank order) and returns 0; any other
 *   value makes the solver return HPSI_ESTATE.  The sum must have the same bits on every rank (hpsi_sum_shards does):
 *   the ranks then take the same decisions and issue the same sequence of calls, which a collective needs.  While an
 *   exchange is set, hpsi_davidson reads each iteration's scalars after its orthogonalisation instead of beside it, so that
 *   the decision never depends on timing.  hpsi_apply / hpsi_diagonal themselves never call fn.
 * fn = NULL removes the hook.  `user` is BORROWED.  Not called for plans without it: single-GPU behaviour is unchanged. */
typedef int (*hpsi_exchange_fn)(void* user, const double* v_dev, double* w_dev, int64_t n, int32_t n_vectors, int64_t ld,
                                void* cuda_stream);
int hpsi_set_exchange(hpsi_plan_t* plan, hpsi_exchange_fn fn, void* user);

/* hpsi_apply with a CUDA event between its kernels: ms_host (HOST, 4 floats) receives the device time of
 * [prep, first-GEMM kernel, second-GEMM kernel, reduce].  Synchronises the stream.  For bench.py's roofline object. */
int hpsi_apply_profiled(hpsi_plan_t* plan, const double* psi_dev, double* out_dev, void* cuda_stream, float* ms_host);

/* Same result through HOST buffers: copies psi to the device, applies, copies out back, synchronises the stream.
 * (End-to-end entry point; operators stay resident in the bound arenas.) */
int hpsi_apply_host(hpsi_plan_t* plan, const double* psi_host, double* out_host, void* cuda_stream);

/* diag(H) on the psi layout (reading A21): diag[l][x,y] = sum over tasks whose A and B blocks are both
 * sector-diagonal of c_t * A[x,x] * B[y,y].  diag_dev: DEVICE, psi_length doubles.  Enqueue only. */
int hpsi_diagonal(hpsi_plan_t* plan, double* diag_dev, void* cuda_stream);

/* Step 8: Davidson-Liu, lowest eigenpair, single root (PAPER.md:62 names the method; A21 gives the
 * algorithm).  All O(psi_length) work and the small subspace eigenproblem run on the device; the host reads back
 * one residual norm per iteration to test convergence.  If the preconditioned correction vanishes under
 * Gram-Schmidt (||s|| < 1e-14; an operator with a diagonal block) while the residual is above tol, the residual itself is
 * taken (reading A21c); the solver stops unconverged only if that vanishes too.  A start vector that already is the
 * eigenvector converges after one mat-vec (converged = 1, residual = 0). */
typedef struct {
  double tol;            /* stop when ||H x - theta x|| <= tol                 (default 1e-8) */
  int32_t max_iter;      /* max matrix-vector products                          (default 200)  */
  int32_t m_max;         /* max subspace dimension before restart, 2..32        (default 16)   */
  int32_t precondition;  /* 1: s = r / (diag(H) - theta) with guard; 0: s = r   (default 1)    */
} hpsi_davidson_params_t;

typedef struct {
  int32_t n_matvec;      /* hpsi_apply calls made                                             */
  int32_t converged;     /* 1 if residual <= tol                                              */
  double residual;       /* last ||H x - theta x||                                            */
} hpsi_davidson_info_t;

/* psi_inout_dev: DEVICE, psi_length doubles; in = start vector (any non-zero), out = normalised Ritz vector.
 * eig_host: HOST, receives theta.  params may be NULL (defaults); info may be NULL.  Synchronises the stream. */
int hpsi_davidson(hpsi_plan_t* plan, double* psi_inout_dev, double* eig_host,
                  const hpsi_davidson_params_t* params, hpsi_davidson_info_t* info, void* cuda_stream);

/* Multi-root variant (SURVEY.md 8(f)-4 "a multi-root / Lanczos variant"; reading A21b): block Davidson-Liu for
 * the n_roots lowest eigenpairs.  Per iteration the k lowest Ritz pairs of G = V^T H V are taken, and for every root whose
 * residual exceeds tol a preconditioned correction vector is orthogonalised (twice) against the basis and appended; the
 * new vectors are multiplied by H in one batched pass over the operators (hpsi_apply_multi) when the plan was built with
 * hpsi_plan_options_t.n_vectors > 1, else one hpsi_apply each.  The basis restarts from the k Ritz vectors when it would
 * outgrow m_max (2 n_roots <= m_max <= 32).  max_iter bounds the mat-vecs.
 *   psi_inout_dev  DEVICE, n_roots vectors `ld` doubles apart (ld >= psi_length): in = start vectors (linearly
 *                  independent), out = orthonormal Ritz vectors, ascending eigenvalue
 *   eig_host       HOST, n_roots doubles;  residual_host: HOST or NULL, n_roots doubles ||H x_i - theta_i x_i||
 *   info           n_matvec, converged (every root <= tol), residual (the largest)
 * Synchronises the stream once per iteration. */
int hpsi_davidson_multi(hpsi_plan_t* plan, double* psi_inout_dev, int64_t ld, int32_t n_roots, double* eig_host,
                        double* residual_host, const hpsi_davidson_params_t* params, hpsi_davidson_info_t* info,
                        void* cuda_stream);

/* The other eigensolver PAPER.md:62 names ("the Lanczos or Davidson method"): explicitly restarted Lanczos with full
 * re-orthogonalisation, lowest eigenpair.  Same arguments as hpsi_davidson (params->precondition is ignored, m_max =
 * Krylov vectors kept before a restart from the Ritz vector).  The loop stops on the Lanczos residual estimate
 * beta_j |y_j| <= tol; info->residual is the true ||H x - theta x|| computed with one extra mat-vec, and
 * info->converged says whether it is <= 10 tol.  Synchronises the stream. */
int hpsi_lanczos(hpsi_plan_t* plan, double* psi_inout_dev, double* eig_host,
                 const hpsi_davidson_params_t* params, hpsi_davidson_info_t* info, void* cuda_stream);

/* Operator streaming from HOST memory ("host-device datacommunication ... due to memory
 * limitations"): for operators that do not fit HBM.  terms->a_data / b_data are pinned HOST arenas here
 * (BORROWED, must outlive the object).  The term list is cut, in the order of the terms' arena positions, into windows
 * whose arena ranges fit `window_doubles` (A + B together); the object owns two device staging slots of that size and one
 * plan per window.  hpsi_stream_apply copies window w+1 on an internal copy stream while window w computes on
 * `cuda_stream`; the windows' results add up in window order (deterministic).  out = H psi (overwrite); psi_dev /
 * out_dev: DEVICE.  Enqueue only, but uses a second stream and events, so it is not CUDA-graph capturable.
 * Blocks stored transposed (a_transposed / b_transposed) are supported: an adjoint term that reads its partner's storage
 * lands in its partner's window, so with shared adjoint storage every operator byte crosses the host link once per apply
 * - half the bytes of the materialised form, the one "compression" a Hermitian H offers without touching the FP64
 * entries (PAPER.md:84 names "data compression techniques" without giving one; synthetic N(0,1) entries have no other
 * redundancy). */
typedef struct hpsi_stream hpsi_stream_t;
int hpsi_stream_create(const hpsi_sectors_t* sectors, const hpsi_terms_t* terms_with_host_arenas, int64_t window_doubles,
                       uint32_t flags, hpsi_stream_t** out);
int hpsi_stream_apply(hpsi_stream_t* s, const double* psi_dev, double* out_dev, void* cuda_stream);
/* what: HPSI_Q_PSI_LENGTH, HPSI_Q_USEFUL_FLOPS, HPSI_Q_OPERATOR_BYTES (= bytes copied host->device per apply),
 * HPSI_SQ_N_WINDOWS, HPSI_SQ_STAGING_BYTES; out: HOST int64. */
enum { HPSI_SQ_N_WINDOWS = 100, HPSI_SQ_STAGING_BYTES = 101 };
int hpsi_stream_query(const hpsi_stream_t* s, int what, void* out, size_t bytes);
void hpsi_stream_destroy(hpsi_stream_t* s);

/* ------------------------------------------------------------------------------------------------------------------
 * Site update after the eigen-solve.  PAPER.md:45 names "tensor contraction and matrix
 * factorization" as the two core operations of tensor-network algorithms and PAPER.md:62 the sweep as a "sequence of
 * updates of all tensors", but writes out neither step; DESIGN.md section 9 lists the readings R1-R6.
 *
 *   hpsi_truncate :  the matrix factorisation.  psi is block diagonal over (left sector l, partner r), so its SVD is
 *                    the SVD of every block, psi_l = U_l S_l V_l^T.  The chi_max largest singular values over all
 *                    blocks are kept (ties: the block that comes first in the psi table; values <=
 *                    1e-13 * sigma_max are never kept) and  O_l = the kept columns of U_l  is the new left basis.
 *   hpsi_rotate_* :  the renormalised-operator update  A'_t[l,l'] = O_l^T A_t[l,l'] O_l'  for every block of every
 *                    left operator, on the same grouped DMMA GEMM engine as hpsi_apply.
 *
 * Isometry layout ("ot", used by both): for l = 0..n_sectors-1 ascending, O_l^T as a dense chi_l x d_l row-major
 * matrix (row a = the a-th kept left singular vector), concatenated; sum_l chi_l d_l doubles.
 * ------------------------------------------------------------------------------------------------------------------ */

/* One-sided block Jacobi SVD (Hestenes rotations, applied 32 rows at a time on the FP64 tensor pipe) of every psi block
 * of `plan`, on the device, then the global selection on the host.
 *   psi_dev        DEVICE, psi_length doubles (not modified)
 *   side           HPSI_SIDE_LEFT: new LEFT basis, O_l = kept left singular vectors (a right-moving sweep);
 *                  HPSI_SIDE_RIGHT: new RIGHT basis, O_r = kept right singular vectors of the block whose right
 *                  sector is r (a left-moving sweep) - "left" below then reads "right", d_left reads d_right
 *   chi_max        number of singular values to keep over all blocks (>= 0)
 *   eps_discard    if >= 0: keep only as many of them as it takes for the discarded weight to be <= eps_discard
 *                  (the paper quotes its results by "truncation error"); < 0: keep chi_max
 *   ot_dev         DEVICE, receives the isometries in the layout above; capacity >= HPSI_Q_ISO_CAPACITY doubles
 *                  (HPSI_Q_ISO_CAPACITY_RIGHT for the right side)
 *   chi_host       HOST, int32[n_left] (n_right for the right side): kept states per sector (0 without a psi block)
 *   sigma_host     HOST or NULL, psi-rows doubles (HPSI_Q_PSI_ROWS = sum of d_left over the psi blocks): for every psi
 *                  block in table order its d_left values, descending; entries past min(d_left, d_right) are 0
 *   discarded_host HOST or NULL: sum of sigma^2 over everything not kept
 * Synchronises the stream (chi is needed on the host).  Deterministic (fixed rotation order; the only atomic is the
 * sweep's rotation counter, which steers nothing but the stop test).  Any block size is accepted.
 * Errors: EINVAL (null / negative arguments), ESTATE (host-only plan, or no convergence in 60 sweeps), ENOMEM, ECUDA. */
#define HPSI_SIDE_LEFT  0
#define HPSI_SIDE_RIGHT 1
int hpsi_truncate(hpsi_plan_t* plan, const double* psi_dev, int32_t side, int32_t chi_max, double eps_discard,
                  double* ot_dev, int32_t* chi_host, double* sigma_host, double* discarded_host, void* cuda_stream);

/* hpsi_truncate for callers that must not allocate device memory (code that may not call cudaMalloc: tight serving
 * loops, harnesses that forbid it).  Same arguments, same steps, same results as hpsi_truncate; the device buffers
 * (working matrices, singular values, tables) live in ONE file-scope `static __device__` array of
 * HPSI_TRUNCATE_STATIC_BYTES instead of the plan's lazily grown cudaMalloc block.  The call makes no cudaMalloc /
 * cudaFree and calls no library routine that allocates; the array's device address is taken once per device
 * (cudaGetSymbolAddress, with that device current - call with the plan's device current).
 *   Limit:    a plan whose psi needs more scratch than the array holds is rejected with EINVAL and a message naming
 *             both sizes (roughly 16 * sum over psi blocks of min(d_l, d_r) * (d_l + d_r) bytes: D = 1024 fits, D = 4096
 *             does not).  Every GPU that loads the library holds the array until the process exits.
 *   Sharing:  every call on a device - any plan, any stream, any thread - uses the same array, which keeps the last
 *             call's contents.  Nothing in it has to start at zero except the per-sweep rotation flag, which the call
 *             clears itself.  Calls that overlap on the GPU race: serialise them (hpsi_truncate has one buffer per plan).
 * Synchronises the stream like hpsi_truncate (chi is needed on the host), so it is not CUDA-graph capturable.
 * Errors: as hpsi_truncate, without ENOMEM. */
#define HPSI_TRUNCATE_STATIC_BYTES (32u << 20)
int hpsi_truncate_static(hpsi_plan_t* plan, const double* psi_dev, int32_t side, int32_t chi_max, double eps_discard,
                         double* ot_dev, int32_t* chi_host, double* sigma_host, double* discarded_host, void* cuda_stream);

typedef struct hpsi_rotate hpsi_rotate_t;   /* opaque; owns the schedule, the workspace (padded isometries, T^T) */

/* Plan the update of `n_blocks` operator blocks of one side.  d / chi: HOST int32[n_sectors], enlarged and kept
 * dimensions (0 <= chi <= d; chi = 0 removes the sector: blocks touching it produce nothing).  blocks: HOST
 * descriptors as in hpsi_terms_t (copied); a_data_dev: DEVICE arena, BORROWED (must outlive the object; not modified);
 * a_len: arena length in doubles (validation; 0 = unknown).  flags: HPSI_PLAN_HOST_ONLY (schedule only, for
 * hpsi_rotate_query / hpsi_rotate_debug_interpret).  The TMA path needs even ld / offset and a 16-byte aligned arena,
 * otherwise the 8-byte cp.async variant of the kernels runs. */
int hpsi_rotate_plan(int32_t n_sectors, const int32_t* d, const int32_t* chi, int64_t n_blocks,
                     const hpsi_opblock_t* blocks, const double* a_data_dev, int64_t a_len, uint32_t flags,
                     hpsi_rotate_t** out);

/* out_dev (DEVICE, HPSI_RQ_OUT_LENGTH doubles) receives every A' block in the plan-dictated layout that
 * HPSI_RQ_OUT_BLOCKS describes (ld = chi[col] rounded up to 4, offsets multiples of 4: directly usable as the operator
 * arena of the next hpsi_plan).  ot_dev: DEVICE isometries (layout above, HPSI_RQ_ISO_LENGTH doubles).  Padding
 * elements of out_dev are not written.  Enqueue only, CUDA-graph capturable, bitwise reproducible. */
int hpsi_rotate_apply(hpsi_rotate_t* r, const double* ot_dev, double* out_dev, void* cuda_stream);
/* same with CUDA events between the kernels: ms_host (HOST, 3 floats) = [isometry copy, first GEMM, second GEMM] */
int hpsi_rotate_apply_profiled(hpsi_rotate_t* r, const double* ot_dev, double* out_dev, void* cuda_stream, float* ms_host);

enum {
  HPSI_RQ_OUT_LENGTH = 0,    /* int64: doubles in the output arena                                               */
  HPSI_RQ_OUT_BLOCKS = 1,    /* hpsi_opblock_t[n_blocks]: descriptor of A'_i for input block i (same term/row/col);
                                a block that vanished (chi[row] == 0 or chi[col] == 0) has ld = 0, offset = -1     */
  HPSI_RQ_ISO_LENGTH = 2,    /* int64: sum_l chi_l d_l                                                            */
  HPSI_RQ_USEFUL_FLOPS = 3,  /* int64: sum over surviving blocks of 2 d_l d_l' chi_l' + 2 chi_l d_l chi_l'        */
  HPSI_RQ_ALGO_BYTES = 4,    /* int64: 8 * (d_l d_l' read + chi_l chi_l' written) over surviving blocks           */
  HPSI_RQ_WORKSPACE_BYTES = 5,
  HPSI_RQ_N_UNITS_1 = 6,     /* int64: CTA work units of the first / second GEMM launch                           */
  HPSI_RQ_N_UNITS_2 = 7,
  HPSI_RQ_ALIGNED16 = 8,     /* int64: 1 if the TMA staging path is used                                          */
  HPSI_RQ_INTERMEDIATE_BYTES = 9 /* int64: bytes of T^T written by the first GEMM (and read by the second)        */
};
int hpsi_rotate_query(const hpsi_rotate_t* r, int what, void* out, size_t bytes);
void hpsi_rotate_destroy(hpsi_rotate_t* r);
/* test entry point: walks the device schedule of the update with naive loops on the HOST (a_host: the arena,
 * ot_host: isometries, out_host: HPSI_RQ_OUT_LENGTH doubles) */
int hpsi_rotate_debug_interpret(const hpsi_rotate_t* r, const double* a_host, const double* ot_host, double* out_host);

/* test entry point: the subspace eigensolver of hpsi_davidson / hpsi_lanczos (k = 1: tridiagonalisation + bisection +
 * inverse iteration by one warp, with the Jacobi solver as fallback; k > 1: the Jacobi solver) on ONE symmetric matrix.
 * g_host: HOST, j x j row-major, 1 <= j <= 32; theta_host: HOST, k values ascending; y_host: HOST, k x j (row r = the
 * r-th eigenvector); fell_back_host: HOST or NULL, 1 if the k = 1 path failed its own check and the Jacobi solver ran.
 * Allocates and frees device memory, synchronises the device. */
int hpsi_debug_small_eig(const double* g_host, int32_t j, int32_t k, double* theta_host, double* y_host,
                         int32_t* fell_back_host);

/* hpsi_query items.  `out` is HOST; `bytes` must be >= the item's size (else EINVAL). */
enum {
  HPSI_Q_PSI_LENGTH = 0,     /* int64: doubles in psi / out                                                  */
  HPSI_Q_N_PSI_BLOCKS = 1,   /* int64                                                                        */
  HPSI_Q_PSI_BLOCKS = 2,     /* hpsi_psi_block_t[n_psi_blocks]                                               */
  HPSI_Q_N_TASKS = 3,        /* int64: realisable (term, A block, B block) triples                            */
  HPSI_Q_USEFUL_FLOPS = 4,   /* int64: sum over tasks of min(2 m n'(k+n), 2 k n(n'+m))  (A18)        */
  HPSI_Q_ISSUED_FLOPS = 5,   /* int64: flops of the DMMA instructions the schedule issues (8x8x4 padding incl.) */
  HPSI_Q_OPERATOR_BYTES = 6, /* int64: 8 * (m k + n n') summed over tasks (bytes streamed once per apply)     */
  HPSI_Q_WORKSPACE_BYTES = 7,/* int64: device workspace the plan owns                                         */
  HPSI_Q_N_GROUPS = 8,       /* int64: (source block, destination block) groups                               */
  HPSI_Q_N_P1_UNITS = 9,     /* int64: CTA work units of the first-GEMM kernel                                */
  HPSI_Q_N_P2_UNITS = 10,    /* int64: CTA work units of the second-GEMM kernel                               */
  HPSI_Q_N_ORDER1_TASKS = 11,/* int64: tasks scheduled as (A psi) B^T                                         */
  HPSI_Q_LAUNCHES_PER_APPLY = 12, /* int64: kernels hpsi_apply enqueues                                       */
  HPSI_Q_ALIGNED16 = 13,     /* int64: 1 if the TMA staging path is used (16-byte aligned rows)              */
  HPSI_Q_INTERMEDIATE_BYTES = 14, /* int64: bytes of first-GEMM results written (and read back) per apply     */
  HPSI_Q_ISSUED_FLOPS_P1 = 15,    /* int64: first-GEMM share of HPSI_Q_ISSUED_FLOPS                           */
  HPSI_Q_TASKS = 16,         /* hpsi_task_t[n_tasks], in schedule order                                      */
  HPSI_Q_USEFUL_FLOPS_P1 = 17,/* int64: first-GEMM share of HPSI_Q_USEFUL_FLOPS                                */
  HPSI_Q_CRITICAL_FLOPS = 18, /* int64: like ISSUED_FLOPS, but every CTA counted as 4 x its heaviest warp (what warp imbalance costs) */
  HPSI_Q_PSI_ROWS = 19,      /* int64: sum of d_left over the psi blocks (length of hpsi_truncate's sigma_host)  */
  HPSI_Q_ISO_CAPACITY = 20,  /* int64: sum of min(d_left, d_right) * d_left over the psi blocks (ot_dev capacity) */
  HPSI_Q_SVD_SWEEPS = 21,    /* int64: Jacobi sweeps of the last hpsi_truncate on this plan                      */
  HPSI_Q_SVD_LAUNCHES = 22,  /* int64: kernels it launched                                                       */
  HPSI_Q_PSI_COLS = 23,      /* int64: sum of d_right over the psi blocks (sigma_host length for HPSI_SIDE_RIGHT)  */
  HPSI_Q_ISO_CAPACITY_RIGHT = 24, /* int64: sum of min(d_left, d_right) * d_right over the psi blocks             */
  HPSI_Q_N_FUSED_UNITS = 25, /* int64: CTA work units of the fused kernel (both GEMMs of a task in one CTA)       */
  HPSI_Q_N_FUSED_TASKS = 26, /* int64: tasks whose intermediate never leaves the chip                             */
  HPSI_Q_TUNING = 27,        /* int64[3]: schedule knobs the plan was built with (hpsi_plan_options_t): first-GEMM K-tiles
                                per CTA, second-GEMM waves, least DMMA count per second-GEMM CTA                    */
  HPSI_Q_PREFERRED_LAYOUT = 28, /* hpsi_layout_t: the operator-arena layout rule (what hpsi_layout_blocks applies)    */
  HPSI_Q_N_TERMS_PLANNED = 29,  /* int64: terms of this plan's shard (= n_terms without hpsi_plan_options_t.shard_of_term) */
  HPSI_Q_N_VECTORS = 30         /* int64: vectors the plan was laid out for (hpsi_plan_options_t.n_vectors, at least 1)     */
};

/* Layout rule of the operator arenas.  A block's rows are `stored columns` doubles long (d[col], or
 * d[row] when the block is flagged transposed) with leading dimension ld. */
typedef struct {
  int32_t ld_multiple;           /* preferred: ld a multiple of this many doubles (4: rows start on 32-byte L2 sectors) */
  int32_t offset_multiple;       /* preferred: block offsets a multiple of this many doubles (4)                       */
  int32_t tma_ld_multiple;       /* required for the TMA staging path: ld and offset multiples of this (2 = 16 bytes);  */
  int32_t tma_offset_multiple;   /*   anything else runs the 8-byte cp.async kernels (correct, slower)                  */
  int32_t arena_align_bytes;     /* required for the TMA path: arena base address alignment (16)                        */
  int32_t transposed_pad_rows;   /* tiles of a plan with transposed blocks are padded to this many rows (8, as plain plans) */
} hpsi_layout_t;

typedef struct {
  int32_t left, right;   /* sector indices                     */
  int32_t rows, cols;    /* d_left[left], d_right[right]       */
  int64_t offset;        /* start in psi, in doubles           */
} hpsi_psi_block_t;

typedef struct {
  int32_t term, a_block, b_block;   /* indices into the term list's a_blocks / b_blocks            */
  int32_t src_left, dst_left;       /* psi blocks (by left sector) read / written                  */
  int32_t order;                    /* 1 = (A psi) B^T, 2 = A (psi B^T)                            */
} hpsi_task_t;

int hpsi_query(const hpsi_plan_t* plan, int what, void* out, size_t bytes);

void hpsi_destroy(hpsi_plan_t* plan);

const char* hpsi_last_error(void);

/* ---- debug / test entry points (HOST memory only; run the *device schedule* with naive loops on the CPU) ----
 * hpsi_debug_interpret executes exactly the work-unit tables the kernels consume (prep, first GEMM units,
 * second GEMM units, ordered reduce) so that the planner can be verified on a box without a GPU.
 * a_host / b_host are HOST copies of the arenas, psi_host / out_host HOST vectors of psi_length doubles. */
int hpsi_debug_interpret(const hpsi_plan_t* plan, const double* a_host, const double* b_host,
                         const double* psi_host, double* out_host);
/* the same for n_vectors vectors of a batched plan, psi_length doubles apart in psi_host / out_host */
int hpsi_debug_interpret_multi(const hpsi_plan_t* plan, const double* a_host, const double* b_host,
                               const double* psi_host, double* out_host, int32_t n_vectors);

#ifdef __cplusplus
}
#endif
#endif /* HPSI_H_ */
