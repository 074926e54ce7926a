/*
 * ORACLE - TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain CPU definition of the hot path of two-site QC-DMRG named by BASELINE.json `north_star`:
 *
 *     psi'(l,r) = sum_t  c_t * A_t(l,l') * psi(l',r') * B_t(r,r')^T            (north_star)
 *
 * i.e. the matrix-vector product inside the "large hermitian eigenvalue problem" that each DMRG
 * tensor update solves "using e.g. the Lanczos or Davidson method" ("Numerical
 * procedure").  The paper never writes the product out; the formula, the block-sparse sector form
 * and the index conventions are BASELINE.json's, with the readings listed in DESIGN.md (A1-A3):
 * real FP64 (Fig. 1 "FP64"), plain transpose, out[x,y] = sum_{x',y'} A[x,x'] psi[x',y'] B[y,y'].
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use this
 * file.  It shares no code, header, table or ordering with paper_2407_07411_b200/ (the CUDA path):
 * always the (A psi) B^T order, naive loops, one writer per output element, loop order = order of the additions into
 * an output element.  One exception, stated here because it is not "as written": the inner dot product over y' of the
 * second product carries `omp simd reduction(+)`, so the compiler may add it up as a few lane-wise partial sums (still
 * deterministic for a given build; the difference is at rounding level, far below the 1e-12 bar).
 *
 * Pins (tests/test_oracle_pins.py): brute-force Kronecker expansion, Hermiticity, single-block = A@psi@B.T,
 * closed forms (identity, rank-1, linearity, power-of-two scaling), Hubbard dimer / 4-site chain energies.
 * Not pinned (needs the paper's integrals): anything about SU(2) recoupling or real-molecule energies -
 * "parity unpinned" for those, and they are out of scope.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {            /* same 24-byte record the boundary uses for one dense operator block */
  int32_t term, row, col, ld;
  int64_t offset;
} oracle_opblock_t;

int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* Step 1 (reading A6/A22): for each left sector i ascending, the unique right sector j
 * with q_left[i] + q_right[j] == target; psi block i is d_left[i] x d_right[j], row-major, appended.
 * partner[i] = j or -1; offset[i] = start of block i in the psi vector (or -1).  Returns psi length. */
int64_t oracle_psi_table(int32_t n_left, int32_t n_right, const int32_t* q_left, const int32_t* q_right,
                         const int32_t* d_left, const int32_t* d_right, const int32_t* target,
                         int32_t* partner, int64_t* offset) {
  int64_t len = 0;
  for (int32_t i = 0; i < n_left; ++i) {
    partner[i] = -1;
    offset[i] = -1;
    for (int32_t j = 0; j < n_right; ++j) {
      if (q_left[2 * i] + q_right[2 * j] == target[0] && q_left[2 * i + 1] + q_right[2 * j + 1] == target[1]) {
        partner[i] = j;
        offset[i] = len;
        len += (int64_t)d_left[i] * d_right[j];
        break;
      }
    }
  }
  return len;
}


/* Order-preserving index of the descriptors of each term: idx[start[t] .. start[t+1]) lists, in the order
 * given, the positions of the blocks with .term == t (descriptors may arrive in any order). */
static int term_index(int32_t n_terms, int64_t n, const oracle_opblock_t* blk, int64_t** start_out,
                      int64_t** idx_out) {
  int64_t* start = (int64_t*)calloc((size_t)n_terms + 2, sizeof(int64_t));
  int64_t* idx = (int64_t*)malloc(sizeof(int64_t) * (size_t)(n > 0 ? n : 1));
  if (!start || !idx) return -1;
  for (int64_t i = 0; i < n; ++i)
    if (blk[i].term >= 0 && blk[i].term < n_terms) start[blk[i].term + 1]++;
  for (int32_t t = 0; t < n_terms; ++t) start[t + 1] += start[t];
  int64_t* fill = (int64_t*)malloc(sizeof(int64_t) * ((size_t)n_terms + 1));
  if (!fill) return -1;
  memcpy(fill, start, sizeof(int64_t) * ((size_t)n_terms + 1));
  for (int64_t i = 0; i < n; ++i)
    if (blk[i].term >= 0 && blk[i].term < n_terms) idx[fill[blk[i].term]++] = i;
  free(fill);
  *start_out = start;
  *idx_out = idx;
  return 0;
}

/* out = H psi, the plain definition evaluated blockwise (SURVEY.md 8(c) "Oracle loop"):
 *   out[:] = 0
 *   for t: for a in A-blocks of t (row l, col l'): for b in B-blocks of t (row r, col r'):
 *     if (l',r') and (l,r) are psi blocks:
 *        T[x,y']   = sum_{x'} a[x,x'] psi_{l'}[x',y']
 *        out_l[x,y] += c_t * sum_{y'} T[x,y'] b[y,y']
 * Blocks of one term are looked up by scanning the descriptor arrays in the order given.
 * OpenMP is over the rows x of one task only, so every output element has one writer and the order of the
 * task contributions added into it is the loop order above (inside one contribution the y' dot product is a simd
 * reduction, see the file header).  Returns 0, or -1 on allocation failure. */
int oracle_apply(int32_t n_left, int32_t n_right, const int32_t* q_left, const int32_t* q_right,
                 const int32_t* d_left, const int32_t* d_right, const int32_t* target,
                 int32_t n_terms, const double* coef,
                 int64_t n_a, const oracle_opblock_t* a_blocks, const double* a_data,
                 int64_t n_b, const oracle_opblock_t* b_blocks, const double* b_data,
                 const double* psi, double* out) {
  int32_t* partner = (int32_t*)malloc(sizeof(int32_t) * (size_t)(n_left > 0 ? n_left : 1));
  int64_t* offset = (int64_t*)malloc(sizeof(int64_t) * (size_t)(n_left > 0 ? n_left : 1));
  if (!partner || !offset) return -1;
  int64_t len = oracle_psi_table(n_left, n_right, q_left, q_right, d_left, d_right, target, partner, offset);
  memset(out, 0, sizeof(double) * (size_t)len);
  int32_t maxr = 1;
  for (int32_t j = 0; j < n_right; ++j) if (d_right[j] > maxr) maxr = d_right[j];
  int nthr = oracle_num_threads();
  double* scratch = (double*)malloc(sizeof(double) * (size_t)maxr * (size_t)nthr);
  if (!scratch) return -1;

  int64_t *sa, *ia_of, *sb, *ib_of;
  if (term_index(n_terms, n_a, a_blocks, &sa, &ia_of) || term_index(n_terms, n_b, b_blocks, &sb, &ib_of)) return -1;

  for (int32_t t = 0; t < n_terms; ++t) {
    const double c = coef[t];
    for (int64_t pa = sa[t]; pa < sa[t + 1]; ++pa) {
      const int64_t ia = ia_of[pa];
      const int32_t l = a_blocks[ia].row, lp = a_blocks[ia].col;
      if (partner[l] < 0 || partner[lp] < 0) continue;
      for (int64_t pb = sb[t]; pb < sb[t + 1]; ++pb) {
        const int64_t ib = ib_of[pb];
        const int32_t r = b_blocks[ib].row, rp = b_blocks[ib].col;
        if (partner[lp] != rp || partner[l] != r) continue;
        const int32_t m = d_left[l], k = d_left[lp], np_ = d_right[rp], n = d_right[r];
        const double* A = a_data + a_blocks[ia].offset;  const int64_t lda = a_blocks[ia].ld;
        const double* B = b_data + b_blocks[ib].offset;  const int64_t ldb = b_blocks[ib].ld;
        const double* P = psi + offset[lp];               /* k  x n' */
        double* O = out + offset[l];                      /* m  x n  */
#pragma omp parallel for schedule(static)
        for (int32_t x = 0; x < m; ++x) {
#ifdef _OPENMP
          double* T = scratch + (size_t)omp_get_thread_num() * (size_t)maxr;
#else
          double* T = scratch;
#endif
          for (int32_t yp = 0; yp < np_; ++yp) T[yp] = 0.0;
          for (int32_t xp = 0; xp < k; ++xp) {
            const double axx = A[x * lda + xp];
            const double* prow = P + (int64_t)xp * np_;
            for (int32_t yp = 0; yp < np_; ++yp) T[yp] += axx * prow[yp];
          }
          for (int32_t y = 0; y < n; ++y) {
            const double* brow = B + y * ldb;
            double s = 0.0;
#pragma omp simd reduction(+ : s)
            for (int32_t yp = 0; yp < np_; ++yp) s += T[yp] * brow[yp];
            O[(int64_t)x * n + y] += c * s;
          }
        }
      }
    }
  }
  free(sa); free(ia_of); free(sb); free(ib_of);
  free(scratch);
  free(partner);
  free(offset);
  return 0;
}

/* Single output elements of H psi, one by one (used where a whole apply is too slow: D=8192):
 *   vals[s] += sum over tasks (t,a,b) writing block sample_left[s]:
 *                c_t * sum_{x'} a[x,x'] * ( sum_{y'} psi_{l'}[x',y'] b[y,y'] ),   x = sample_x[s], y = sample_y[s]
 * ACCUMULATES into vals (caller zeroes), so that a caller may stream disjoint term subsets through it.
 * Descriptor offsets are relative to a_data/b_data as passed. */
int oracle_apply_samples(int32_t n_left, int32_t n_right, const int32_t* q_left, const int32_t* q_right,
                         const int32_t* d_left, const int32_t* d_right, const int32_t* target,
                         int32_t n_terms, const double* coef,
                         int64_t n_a, const oracle_opblock_t* a_blocks, const double* a_data,
                         int64_t n_b, const oracle_opblock_t* b_blocks, const double* b_data,
                         const double* psi, int32_t n_samples, const int32_t* sample_left,
                         const int32_t* sample_x, const int32_t* sample_y, double* vals) {
  int32_t* partner = (int32_t*)malloc(sizeof(int32_t) * (size_t)(n_left > 0 ? n_left : 1));
  int64_t* offset = (int64_t*)malloc(sizeof(int64_t) * (size_t)(n_left > 0 ? n_left : 1));
  if (!partner || !offset) return -1;
  oracle_psi_table(n_left, n_right, q_left, q_right, d_left, d_right, target, partner, offset);
  int64_t *sb, *ib_of;
  if (term_index(n_terms, n_b, b_blocks, &sb, &ib_of)) return -1;
#pragma omp parallel for schedule(dynamic, 1)
  for (int32_t s = 0; s < n_samples; ++s) {
    const int32_t l = sample_left[s], x = sample_x[s], y = sample_y[s];
    if (partner[l] < 0) continue;
    const int32_t r = partner[l];
    double acc = 0.0;
    for (int64_t ia = 0; ia < n_a; ++ia) {
      if (a_blocks[ia].row != l) continue;
      const int32_t t = a_blocks[ia].term, lp = a_blocks[ia].col;
      if (partner[lp] < 0 || t < 0 || t >= n_terms) continue;
      for (int64_t pb = sb[t]; pb < sb[t + 1]; ++pb) {
        const int64_t ib = ib_of[pb];
        if (b_blocks[ib].row != r || b_blocks[ib].col != partner[lp]) continue;
        const int32_t k = d_left[lp], np_ = d_right[partner[lp]];
        const double* A = a_data + a_blocks[ia].offset + (int64_t)x * a_blocks[ia].ld;
        const double* B = b_data + b_blocks[ib].offset + (int64_t)y * b_blocks[ib].ld;
        const double* P = psi + offset[lp];
        double tsum = 0.0;
        for (int32_t xp = 0; xp < k; ++xp) {
          double u = 0.0;
          for (int32_t yp = 0; yp < np_; ++yp) u += P[(int64_t)xp * np_ + yp] * B[yp];
          tsum += A[xp] * u;
        }
        acc += coef[t] * tsum;
      }
    }
    vals[s] += acc;
  }
  free(sb); free(ib_of);
  free(partner);
  free(offset);
  return 0;
}
