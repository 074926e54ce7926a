// Host planner: sector table + term list -> flat device schedule.
//
//  1. psi block table: left sector i pairs with the unique right sector j with q_left[i]+q_right[j]==Q*.
//  2. task enumeration: (t, A block l<-l', B block r<-r') with (l',r') and (l,r) both psi blocks.
//  3. order choice per task by flops: f1 = 2 m n'(k+n) for (A psi)B^T, f2 = 2 k n(n'+m) for A(psi B^T)
//     (north_star: "orders each term as (A psi)B^T or A(psi B^T) by flop count"); tie -> order 1.
//  4. grouping: tasks sorted by (destination block, source block, term).  A (source,destination) group shares
//     all four dims; its first GEMMs are stacked into one tall GEMM, and all groups of one destination form
//     the K dimension of that block's second GEMM ("groups all tasks that write one output block so accumulation
//     stays on-chip with no global atomics").  K is cut into chunks of roughly equal DMMA count (split-K partials,
//     reduced in a fixed order), output blocks into <=64x64 tiles with an even split in units of 8x8 fragments.
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <numeric>
#include <unordered_map>

#include "plan.h"

namespace hpsi {

// Split of a dimension into tiles of at most max_frags fragments.  Inside a CTA the tile is cut again between the
// consumer warps (2 or 4 ways per dimension), so tile sizes are multiples of `unit` fragments wherever possible and
// only the last tile takes the remainder: a tile with an odd fragment count leaves a warp row (or column) short and
// the whole CTA waits for its heaviest warp.  (cyp, 64x64 tiles: issued / critical-path DMMA 0.865 with an even
// split, 0.954 with unit 2.)
std::vector<Tile1D> split_dim(int64_t n, int max_frags, int unit) {
  std::vector<Tile1D> out;
  if (n <= 0) return out;
  const int64_t F = (n + 7) / 8;
  const int64_t nt = (F + max_frags - 1) / max_frags;
  std::vector<int64_t> fr(nt);
  const int64_t P = F / unit, base = P / nt, rem = P % nt;
  for (int64_t i = 0; i < nt; ++i) fr[i] = unit * (base + (i < rem ? 1 : 0));
  fr[nt - 1] += F - unit * P;                      // the last tile is the smallest (or tied): it takes the remainder
  if (*std::max_element(fr.begin(), fr.end()) > max_frags) {      // cannot happen for unit | max_frags; keep it safe
    const int64_t b2 = F / nt, r2 = F % nt;
    for (int64_t i = 0; i < nt; ++i) fr[i] = b2 + (i < r2 ? 1 : 0);
  }
  int64_t start = 0;
  for (int64_t i = 0; i < nt; ++i) {
    if (fr[i] == 0) continue;
    const int64_t len = std::min<int64_t>(fr[i] * 8, n - start);
    out.push_back({(int)start, (int)len});
    start += fr[i] * 8;
  }
  return out;
}
// rows: up to TILE_M; columns: up to TILE.  Units: half of what the warp grid cuts each dimension into.
std::vector<Tile1D> split_rows(int64_t n) { return split_dim(n, TILE_M / 8, 2); }
std::vector<Tile1D> split_cols(int64_t n) { return split_dim(n, TILE / 8, 2); }
namespace {

int64_t align_up(int64_t x, int64_t a) { return (x + a - 1) / a * a; }

#define FAIL(code, ...)                                   \
  do {                                                    \
    char buf_[512];                                       \
    snprintf(buf_, sizeof buf_, __VA_ARGS__);             \
    *err = buf_;                                          \
    return code;                                          \
  } while (0)

struct RawTask {
  int32_t term, ia, ib, src, dst;   // src/dst = psi block indices
  int32_t ta, tb;                   // A / B block stored transposed
};

}  // namespace

// psi block table alone (step 1): blk_of_left[i] = psi block of left sector i or -1, partner[i] = its right sector
static void psi_pairs(const hpsi_sectors_t* s, std::vector<int>* blk_of_left, std::vector<int>* partner) {
  std::unordered_map<uint64_t, int> right_by_label;
  for (int j = 0; j < s->n_right; ++j)
    right_by_label[((uint64_t)(uint32_t)s->q_right[2 * j] << 32) | (uint32_t)s->q_right[2 * j + 1]] = j;
  blk_of_left->assign(s->n_left, -1);
  partner->assign(s->n_left, -1);
  int nb = 0;
  for (int i = 0; i < s->n_left; ++i) {
    const int32_t wantN = s->target[0] - s->q_left[2 * i], wantS = s->target[1] - s->q_left[2 * i + 1];
    auto it = right_by_label.find(((uint64_t)(uint32_t)wantN << 32) | (uint32_t)wantS);
    if (it == right_by_label.end()) continue;
    (*blk_of_left)[i] = nb++;
    (*partner)[i] = it->second;
  }
}

int term_useful_flops(const hpsi_sectors_t* s, const hpsi_terms_t* t, std::vector<int64_t>* flops, std::string* err) {
  if (!s || !t || !flops) FAIL(HPSI_EINVAL, "null argument");
  const int nL = s->n_left, nR = s->n_right;
  if (nL < 0 || nR < 0 || t->n_terms < 0 || t->n_a < 0 || t->n_b < 0) FAIL(HPSI_EINVAL, "negative count");
  if ((nL > 0 && (!s->q_left || !s->d_left)) || (nR > 0 && (!s->q_right || !s->d_right))) FAIL(HPSI_EINVAL, "null sector arrays");
  if ((t->n_a > 0 && !t->a_blocks) || (t->n_b > 0 && !t->b_blocks)) FAIL(HPSI_EINVAL, "null term arrays");
  std::vector<int> blk_of_left, partner;
  psi_pairs(s, &blk_of_left, &partner);
  flops->assign((size_t)t->n_terms, 0);
  std::unordered_map<uint64_t, int64_t> b_index;
  b_index.reserve((size_t)t->n_b * 2);
  for (int64_t i = 0; i < t->n_b; ++i) {
    const hpsi_opblock_t& e = t->b_blocks[i];
    if (e.term < 0 || e.term >= t->n_terms || e.row < 0 || e.row >= nR || e.col < 0 || e.col >= nR)
      FAIL(HPSI_EINVAL, "B block %lld: term or sector index out of range", (long long)i);
    b_index[((uint64_t)e.term * (uint64_t)nR + (uint64_t)e.row) * (uint64_t)nR + (uint64_t)e.col] = i;
  }
  for (int64_t ia = 0; ia < t->n_a; ++ia) {
    const hpsi_opblock_t& a = t->a_blocks[ia];
    if (a.term < 0 || a.term >= t->n_terms || a.row < 0 || a.row >= nL || a.col < 0 || a.col >= nL)
      FAIL(HPSI_EINVAL, "A block %lld: term or sector index out of range", (long long)ia);
    if (blk_of_left[a.row] < 0 || blk_of_left[a.col] < 0) continue;
    const uint64_t key = ((uint64_t)a.term * (uint64_t)nR + (uint64_t)partner[a.row]) * (uint64_t)nR + (uint64_t)partner[a.col];
    if (b_index.find(key) == b_index.end()) continue;
    const int64_t m = s->d_left[a.row], k = s->d_left[a.col], n = s->d_right[partner[a.row]], np = s->d_right[partner[a.col]];
    (*flops)[a.term] += std::min(2 * m * np * (k + n), 2 * k * n * (np + m));
  }
  return HPSI_OK;
}

int build_schedule(const hpsi_sectors_t* s, const hpsi_terms_t* t, uint32_t flags, int n_sm, const PlanOptions& opt,
                   Schedule* sc, std::string* err) {
  if (!s || !t || !sc) FAIL(HPSI_EINVAL, "null argument");
  const int nL = s->n_left, nR = s->n_right;
  if (nL < 0 || nR < 0) FAIL(HPSI_EINVAL, "negative sector count");
  if ((nL > 0 && (!s->q_left || !s->d_left)) || (nR > 0 && (!s->q_right || !s->d_right)))
    FAIL(HPSI_EINVAL, "null sector arrays");
  if (t->n_terms < 0 || t->n_a < 0 || t->n_b < 0) FAIL(HPSI_EINVAL, "negative term/block count");
  if ((t->n_terms > 0 && !t->coef) || (t->n_a > 0 && !t->a_blocks) || (t->n_b > 0 && !t->b_blocks))
    FAIL(HPSI_EINVAL, "null term arrays");
  if ((flags & HPSI_PLAN_FIXED_ORDER1) && (flags & HPSI_PLAN_FIXED_ORDER2))
    FAIL(HPSI_EINVAL, "both fixed-order flags set");
  if (opt.p1_stages_per_unit < 0 || opt.p2_waves < 0 || opt.p2_min_unit_dmma < 0) FAIL(HPSI_EINVAL, "negative schedule knob");
  if (opt.n_vectors < 0 || opt.n_vectors > 64) FAIL(HPSI_EINVAL, "n_vectors outside 0..64");
  const int nvec = std::max(1, opt.n_vectors);
  sc->nvec = nvec;
  if (nvec > 1 && (flags & HPSI_PLAN_FUSE_ALL)) FAIL(HPSI_EINVAL, "batched plans (n_vectors > 1) do not run the fused kernel");
  // term shard: only the terms with shard_of_term[t] == shard_index are planned; the blocks of every
  // other term are ignored altogether (their descriptors are not validated: the caller's arenas need not hold them)
  auto in_shard = [&](int32_t term) { return !opt.shard_of_term || opt.shard_of_term[term] == opt.shard_index; };
  sc->n_terms_planned = 0;
  for (int32_t term = 0; term < t->n_terms; ++term) sc->n_terms_planned += in_shard(term) ? 1 : 0;

  // ---- validation of the sector table (reading A22: labels unique per side, dims >= 1)
  auto check_side = [&](int n, const int32_t* q, const int32_t* d, const char* side) -> int {
    std::unordered_map<uint64_t, int> seen;
    for (int i = 0; i < n; ++i) {
      if (d[i] < 1) FAIL(HPSI_EINVAL, "%s sector %d has dimension %d < 1", side, i, d[i]);
      uint64_t key = ((uint64_t)(uint32_t)q[2 * i] << 32) | (uint32_t)q[2 * i + 1];
      if (!seen.emplace(key, i).second) FAIL(HPSI_EINVAL, "duplicate %s sector label (%d,%d)", side, q[2 * i], q[2 * i + 1]);
    }
    return HPSI_OK;
  };
  if (int rc = check_side(nL, s->q_left, s->d_left, "left")) return rc;
  if (int rc = check_side(nR, s->q_right, s->d_right, "right")) return rc;

  // ---- step 1: psi block table
  std::unordered_map<uint64_t, int> right_by_label;
  for (int j = 0; j < nR; ++j)
    right_by_label[((uint64_t)(uint32_t)s->q_right[2 * j] << 32) | (uint32_t)s->q_right[2 * j + 1]] = j;
  std::vector<int> blk_of_left(nL, -1), partner(nL, -1);
  sc->blocks.clear();
  int64_t off = 0;
  for (int i = 0; i < nL; ++i) {
    int32_t wantN = s->target[0] - s->q_left[2 * i], wantS = s->target[1] - s->q_left[2 * i + 1];
    auto it = right_by_label.find(((uint64_t)(uint32_t)wantN << 32) | (uint32_t)wantS);
    if (it == right_by_label.end()) continue;
    PsiBlk b{};
    b.left = i;
    b.right = it->second;
    b.rows = s->d_left[i];
    b.cols = s->d_right[it->second];
    b.off = off;
    b.ldp = sector_up(b.cols);
    b.ldt = sector_up(b.rows);
    off += (int64_t)b.rows * b.cols;
    blk_of_left[i] = (int)sc->blocks.size();
    partner[i] = it->second;
    sc->blocks.push_back(b);
  }
  sc->psi_len = off;
  const int nB = (int)sc->blocks.size();
  sc->elem.clear();
  for (int b = 0; b < nB; ++b)
    for (int e0 = 0; e0 < sc->blocks[b].rows * sc->blocks[b].cols; e0 += 256) sc->elem.push_back({b, e0});

  // ---- validation of block descriptors
  sc->aligned16 = true;
  auto check_blocks = [&](int64_t n, const hpsi_opblock_t* blk, const uint8_t* tr, const int32_t* d, int nsec,
                          int64_t arena_len, const char* side) -> int {
    std::unordered_map<uint64_t, int64_t> seen;
    seen.reserve((size_t)n * 2);
    for (int64_t i = 0; i < n; ++i) {
      const hpsi_opblock_t& e = blk[i];
      if (e.term < 0 || e.term >= t->n_terms) FAIL(HPSI_EINVAL, "%s block %lld: term %d out of range", side, (long long)i, e.term);
      if (!in_shard(e.term)) continue;
      if (e.row < 0 || e.row >= nsec || e.col < 0 || e.col >= nsec)
        FAIL(HPSI_EINVAL, "%s block %lld: sector index out of range", side, (long long)i);
      const bool tflag = tr && tr[i];                       // stored as the d[col] x d[row] transpose
      const int srows = tflag ? d[e.col] : d[e.row], scols = tflag ? d[e.row] : d[e.col];
      if (e.ld < scols) FAIL(HPSI_EINVAL, "%s block %lld: ld %d < stored cols %d", side, (long long)i, e.ld, scols);
      if (e.offset < 0) FAIL(HPSI_EINVAL, "%s block %lld: negative offset", side, (long long)i);
      int64_t last = e.offset + (int64_t)(srows - 1) * e.ld + scols;
      if (arena_len > 0 && last > arena_len)
        FAIL(HPSI_EINVAL, "%s block %lld: extends past the arena (%lld > %lld)", side, (long long)i, (long long)last, (long long)arena_len);
      uint64_t key = ((uint64_t)e.term * (uint64_t)nsec + (uint64_t)e.row) * (uint64_t)nsec + (uint64_t)e.col;
      if (!seen.emplace(key, i).second)
        FAIL(HPSI_EINVAL, "%s: two blocks for (term %d, row %d, col %d)", side, e.term, e.row, e.col);
    }
    return HPSI_OK;
  };
  if (int rc = check_blocks(t->n_a, t->a_blocks, t->a_transposed, s->d_left, nL, t->a_len, "A")) return rc;
  if (int rc = check_blocks(t->n_b, t->b_blocks, t->b_transposed, s->d_right, nR, t->b_len, "B")) return rc;

  sc->paired = false;
  if (t->a_transposed) for (int64_t i = 0; i < t->n_a; ++i) if (t->a_transposed[i] && in_shard(t->a_blocks[i].term)) sc->paired = true;
  if (t->b_transposed) for (int64_t i = 0; i < t->n_b; ++i) if (t->b_transposed[i] && in_shard(t->b_blocks[i].term)) sc->paired = true;
  const bool paired = sc->paired;
  if (nvec > 1 && paired) FAIL(HPSI_EINVAL, "batched plans (n_vectors > 1) do not support blocks stored transposed");

  // ---- step 2: task enumeration
  std::unordered_map<uint64_t, int64_t> b_index;
  b_index.reserve((size_t)t->n_b * 2);
  for (int64_t i = 0; i < t->n_b; ++i) {
    const hpsi_opblock_t& e = t->b_blocks[i];
    if (!in_shard(e.term)) continue;
    b_index[((uint64_t)e.term * (uint64_t)nR + (uint64_t)e.row) * (uint64_t)nR + (uint64_t)e.col] = i;
  }
  std::vector<RawTask> raw;
  for (int64_t ia = 0; ia < t->n_a; ++ia) {
    const hpsi_opblock_t& a = t->a_blocks[ia];
    if (!in_shard(a.term)) continue;
    int dst = blk_of_left[a.row], src = blk_of_left[a.col];
    if (dst < 0 || src < 0) continue;
    uint64_t key = ((uint64_t)a.term * (uint64_t)nR + (uint64_t)partner[a.row]) * (uint64_t)nR + (uint64_t)partner[a.col];
    auto it = b_index.find(key);
    if (it == b_index.end()) continue;
    raw.push_back({a.term, (int32_t)ia, (int32_t)it->second, src, dst,
                   (t->a_transposed && t->a_transposed[ia]) ? 1 : 0,
                   (t->b_transposed && t->b_transposed[it->second]) ? 1 : 0});
  }
  // inside a (source, destination) group: tasks with the same storage layout together, then by term
  std::stable_sort(raw.begin(), raw.end(), [](const RawTask& x, const RawTask& y) {
    if (x.dst != y.dst) return x.dst < y.dst;
    if (x.src != y.src) return x.src < y.src;
    if (x.ta != y.ta) return x.ta < y.ta;
    if (x.tb != y.tb) return x.tb < y.tb;
    return x.term < y.term;
  });

  // ---- workspace layout part 1: padded psi and psi^T
  int64_t ws = 0;
  for (auto& b : sc->blocks) {                  // batched plans: the nvec copies one under the other, no padding rows
    b.p_off = ws;
    b.p_vstride = (int64_t)b.rows * b.ldp;
    ws = align_up(ws + nvec * b.p_vstride, 16);
  }
  for (auto& b : sc->blocks) {
    b.t_off = ws;
    b.t_vstride = (int64_t)b.cols * b.ldt;
    ws = align_up(ws + nvec * b.t_vstride, 16);
    sc->max_block_elems = std::max<int32_t>(sc->max_block_elems, b.rows * b.cols);
  }
  sc->maps.clear();
  auto add_map = [&](int base, int64_t moff, int rows, int cols, int ld) -> int32_t {
    sc->maps.push_back({moff, base, rows, cols, ld, TILE, KT});
    return (int32_t)sc->maps.size() - 1;
  };
  // operator block that is an NT operand with op_rows rows and K = op_k columns; stored transposed if tr
  auto add_op_map = [&](int base, int64_t moff, int op_rows, int op_k, int ld, int tr) -> int32_t {
    if (!tr) return add_map(base, moff, op_rows, op_k, ld);
    sc->maps.push_back({moff, base, op_k, op_rows, ld, KT, 8});     // T layout: 8 operand rows (64 bytes) x 16 k per box
    return (int32_t)sc->maps.size() - 1;
  };
  for (auto& b : sc->blocks) {
    b.p_map = add_map(BASE_WS, b.p_off, nvec * b.rows, b.cols, b.ldp);
    b.t_map = add_map(BASE_WS, b.t_off, nvec * b.cols, b.rows, b.ldt);
  }

  // The fused kernel is OFF by default: measured on B200 it loses to the two launches even where every task fits it
  // (cyp-shaped config at D = 1024: 1.83 ms per apply fused, 0.63 ms through the workspace - per segment the first GEMM,
  // a CTA barrier, the shared-memory write, a barrier and the second GEMM run back to back, where the two-launch kernels
  // stream stages without ever draining).  HPSI_PLAN_FUSE_ALL selects it.

  // ---- steps 3+4a: order choice, groups, segs
  sc->segs.clear(); sc->groups.clear(); sc->tasks.clear(); sc->diag.clear();
  sc->useful_flops = sc->useful_flops_p1 = sc->operator_bytes = sc->intermediate_bytes = 0;
  sc->n_order1 = 0;
  std::vector<std::vector<DiagTask>> diag_by_blk(nB);
  for (size_t i = 0; i < raw.size();) {
    size_t j = i;
    while (j < raw.size() && raw[j].dst == raw[i].dst && raw[j].src == raw[i].src) ++j;
    const PsiBlk& S = sc->blocks[raw[i].src];
    const PsiBlk& D = sc->blocks[raw[i].dst];
    const int64_t m = D.rows, n = D.cols, k = S.rows, np = S.cols;
    const int64_t f1 = 2 * m * np * (k + n), f2 = 2 * k * n * (np + m);
    int order = (f2 < f1) ? 2 : 1;
    if (flags & HPSI_PLAN_FIXED_ORDER1) order = 1;
    if (flags & HPSI_PLAN_FIXED_ORDER2) order = 2;
    // the first GEMM's units take [plain | transposed] halves of the group, so its operand's layout is the primary key
    // (the sort above put A's first: right for order 1 only); the second GEMM's runs split at every layout change
    if (order == 2 && paired)
      std::stable_sort(raw.begin() + i, raw.begin() + j, [](const RawTask& x, const RawTask& y) {
        if (x.tb != y.tb) return x.tb < y.tb;
        if (x.ta != y.ta) return x.ta < y.ta;
        return x.term < y.term;
      });
    Group g{};
    g.order = order;
    g.tcount = (int32_t)(j - i);
    g.seg0 = (int32_t)sc->segs.size();
    g.src = raw[i].src;
    g.dst = raw[i].dst;
    if (order == 1) { g.rows = (int32_t)m; g.K1 = (int32_t)k; g.N1 = (int32_t)np; g.ldy1 = S.ldt; g.y1_off = S.t_off; g.y1_map = S.t_map; }
    else            { g.rows = (int32_t)n; g.K1 = (int32_t)np; g.N1 = (int32_t)k; g.ldy1 = S.ldp; g.y1_off = S.p_off; g.y1_map = S.p_map; }
    // Batched plans: the first GEMM's results of the nvec vectors sit side by side in one row, vector v in columns
    // [v N1p, v N1p + N1); N1p is a multiple of the K-tile and the pad columns are never written (the workspace is zeroed
    // at plan time), so a K-tile of the second GEMM never reaches into the next vector.
    g.N1p = nvec > 1 ? (int32_t)align_up(g.N1, KT) : g.N1;
    g.ldw = nvec > 1 ? nvec * g.N1p : sector_up(g.N1);
    // Narrow groups run both GEMMs in one CTA (kernels_fused.cu; north_star: "the intermediate block kept in shared
    // memory or registers between the two GEMMs"): the whole intermediate of a tile fits one operand buffer (N1 <= 64)
    // and the output dimension that would otherwise recompute it is a single tile (order 1: n <= 64, order 2: m <= 64).
    {
      const int64_t other = (order == 1) ? n : m;
      const bool fits = g.N1 <= TILE && other <= TILE && !paired;
      g.fused = (fits && !(flags & HPSI_PLAN_NO_FUSION) && (flags & HPSI_PLAN_FUSE_ALL)) ? 1 : 0;
    }
    g.ws_off = ws;
    const int64_t per_task = g.fused ? 0 : (int64_t)g.rows * g.ldw;
    g.ws_map = g.fused ? -1 : add_map(BASE_WS, ws, (int)((int64_t)g.rows * (j - i)), nvec > 1 ? g.ldw : g.N1, g.ldw);
    for (size_t q = i; q < j; ++q) {
      const hpsi_opblock_t& a = t->a_blocks[raw[q].ia];
      const hpsi_opblock_t& b = t->b_blocks[raw[q].ib];
      Seg sg{};
      // operator blocks as NT operands: A_t is (m x k), B_t is (n x n'); each block belongs to exactly one task
      if (order == 1) {
        sg.p1_off = a.offset; sg.p1_ld = a.ld; sg.p2_off = b.offset; sg.p2_ld = b.ld;
        sg.p1_trans = raw[q].ta; sg.p2_trans = raw[q].tb;
        sg.p1_map = add_op_map(BASE_A, a.offset, (int)m, (int)k, a.ld, raw[q].ta);
        sg.p2_map = add_op_map(BASE_B, b.offset, (int)n, (int)np, b.ld, raw[q].tb);
      } else {
        sg.p1_off = b.offset; sg.p1_ld = b.ld; sg.p2_off = a.offset; sg.p2_ld = a.ld;
        sg.p1_trans = raw[q].tb; sg.p2_trans = raw[q].ta;
        sg.p1_map = add_op_map(BASE_B, b.offset, (int)n, (int)np, b.ld, raw[q].tb);
        sg.p2_map = add_op_map(BASE_A, a.offset, (int)m, (int)k, a.ld, raw[q].ta);
      }
      sg.coef = t->coef[raw[q].term];
      sc->segs.push_back(sg);
      if ((a.offset & 1) || (a.ld & 1) || (b.offset & 1) || (b.ld & 1)) sc->aligned16 = false;
      sc->tasks.push_back({raw[q].term, raw[q].ia, raw[q].ib, S.left, D.left, order});
      sc->useful_flops += std::min(f1, f2);
      sc->useful_flops_p1 += (f2 < f1) ? 2 * k * np * n : 2 * m * k * np;   // first GEMM of the min-flop order
      sc->operator_bytes += 8 * (m * k + n * np);
      if (!g.fused) sc->intermediate_bytes += 8 * (int64_t)g.rows * g.N1;
      if (order == 1) sc->n_order1++;
      if (raw[q].src == raw[q].dst)
        diag_by_blk[raw[q].dst].push_back({a.offset, b.offset, a.ld, b.ld, t->coef[raw[q].term], (int32_t)sc->segs.size() - 1, 0});
    }
    ws = align_up(ws + per_task * g.tcount, 16);
    sc->groups.push_back(g);
    i = j;
  }
  for (int b = 0; b < nB; ++b) {
    sc->blocks[b].diag0 = (int32_t)sc->diag.size();
    sc->diag.insert(sc->diag.end(), diag_by_blk[b].begin(), diag_by_blk[b].end());
    sc->blocks[b].diag1 = (int32_t)sc->diag.size();
  }

  // ---- step 4b: P1 units.  One unit = one tile position of the (rows x N1) intermediate and a range of the group's
  // terms, processed back to back by one CTA (the staging pipeline runs across terms, so the CTA prologue and the
  // load latency are paid once per ~P1_STAGES_PER_UNIT K-tiles instead of once per task).  Column tile fastest, so
  // the tiles that read the same operator rows are adjacent in launch order; groups go heaviest unit first.
  sc->p1.clear();
  sc->issued_flops_p1 = 0;
  sc->critical_flops = 0;
  {
    // ~96 K-tiles per unit, fewer when the whole launch would otherwise be only a few waves of CTAs (small problems)
    int64_t total_stages = 0;
    for (const Group& g : sc->groups)
      if (!g.fused) total_stages += (int64_t)nvec * split_rows(g.rows).size() * split_cols(g.N1).size() * g.tcount * ((g.K1 + KT - 1) / KT);
    const int auto_stages = (int)std::max<int64_t>(12, std::min<int64_t>(96, total_stages / ((int64_t)std::max(n_sm, 1) * 3 * 8)));
    const int P1_STAGES_PER_UNIT = opt.p1_stages_per_unit > 0 ? opt.p1_stages_per_unit : auto_stages;
    sc->tuning[0] = P1_STAGES_PER_UNIT;
    struct GOrder { int64_t cost; int gi; };
    std::vector<GOrder> gorder;
    std::vector<int> g_nt(sc->groups.size());
    for (size_t gi = 0; gi < sc->groups.size(); ++gi) {
      const Group& g = sc->groups[gi];
      if (g.fused) continue;
      const int stages = (g.K1 + KT - 1) / KT;
      int nt = std::max(1, std::min(g.tcount, (P1_STAGES_PER_UNIT + stages - 1) / stages));
      const int nchunk = (g.tcount + nt - 1) / nt;
      nt = (g.tcount + nchunk - 1) / nchunk;                    // even chunks
      g_nt[gi] = nt;
      const int fr = std::min(frags(g.rows), TILE_M / 8), fc = std::min(frags(g.N1), TILE / 8);
      gorder.push_back({(int64_t)fr * fc * ((g.K1 + 3) / 4) * nt, (int)gi});
    }
    std::stable_sort(gorder.begin(), gorder.end(), [](const GOrder& x, const GOrder& y) { return x.cost > y.cost; });
    for (const GOrder& go : gorder) {
      const Group& g = sc->groups[go.gi];
      auto rt = split_rows(g.rows);
      auto ct = split_cols(g.N1);
      const int64_t ks = (g.K1 + 3) / 4;
      const int nt = g_nt[go.gi];
      int tb = 0;                                   // segs [0, tb) have a plainly stored P1 operator block, [tb, tcount) a transposed one
      while (tb < g.tcount && !sc->segs[g.seg0 + tb].p1_trans) ++tb;
      for (int part = 0; part < 2; ++part) {
        const int lo = part ? tb : 0, hi = part ? g.tcount : tb;
        for (int t0 = lo; t0 < hi; t0 += nt) {
          const int t1 = std::min(hi, t0 + nt);
          for (auto& r : rt)
            for (auto& c : ct) {
              const int fm = tile_frags(r.len, paired), fn = tile_frags(c.len, paired);
              int heavy = 0;
              const int32_t grid = best_grid(fm, fn, &heavy, paired);
              for (int v = 0; v < nvec; ++v)            // the vectors of a tile are adjacent: they read the same operator rows
                sc->p1.push_back({go.gi, t0, t1, r.start, r.len, c.start, c.len, grid, part, v});
              sc->issued_flops_p1 += (int64_t)fm * fn * ks * 512 * (t1 - t0);        // flop counts are per vector
              sc->critical_flops += (int64_t)NCONS_WARPS * heavy * ks * 512 * (t1 - t0);
            }
        }
      }
    }
  }

  // ---- step 4c: P2 units.  K-space of destination d = all segs of all groups with dst == d, in seg order.
  // Cost model (used to cut K into chunks and to order the units): a staged K-tile costs the CTA its DMMAs, but never
  // less than STAGE_FLOOR DMMA-equivalents - the barrier round trip and the tile load of a stage take ~500 clk even
  // when a tiny segment (K <= 4 ... 8) or a tiny tile leaves almost nothing to multiply.  Without the floor, units made
  // of thousands of tiny segments ran 20x longer than planned (stress config: SMs active 85 % of the P2 launch).
  constexpr int64_t STAGE_FLOOR = 48;
  auto seg_cost = [&](const Group& g, int64_t tile_frags) {      // one segment on a tile of tile_frags fragments
    const int64_t full = g.N1 / KT, rem = g.N1 % KT;
    int64_t c = full * std::max<int64_t>(4 * tile_frags, STAGE_FLOOR);
    if (rem) c += std::max<int64_t>(((rem + 3) / 4) * tile_frags, STAGE_FLOOR);
    return c;
  };
  // A fused segment (kernels_fused.cu) runs its first GEMM in the same CTA: ceil(K1/16) more stages on the intermediate's tile.
  auto fused_extra = [&](const Group& g, int64_t tile_frags_a) {
    const int64_t full = g.K1 / KT, rem = g.K1 % KT;
    int64_t c = full * std::max<int64_t>(4 * tile_frags_a, STAGE_FLOOR);
    if (rem) c += std::max<int64_t>(((rem + 3) / 4) * tile_frags_a, STAGE_FLOOR);
    return c;
  };
  // pass 0: groups whose intermediate is in the workspace (p2 units); pass 1: fused groups (pf units)
  struct DstInfo { int g0 = 0, g1 = 0; int64_t cost[2] = {0, 0}; int64_t nseg[2] = {0, 0}; int maxf = 0; std::vector<Tile1D> rt, ct; };
  std::vector<DstInfo> dsts(nB);
  int64_t total_cost[2] = {0, 0};
  auto group_seg_cost = [&](const Group& g, int64_t tile_frags_b) {
    int64_t c = seg_cost(g, tile_frags_b);
    if (g.fused) c += fused_extra(g, (int64_t)std::min(frags(g.rows), TILE_M / 8) * frags(g.N1));
    return c;
  };
  {
    size_t gi = 0;
    for (int d = 0; d < nB; ++d) {
      DstInfo& di = dsts[d];
      di.rt = split_rows(sc->blocks[d].rows);
      di.ct = split_cols(sc->blocks[d].cols);
      for (auto& r : di.rt) for (auto& c : di.ct) di.maxf = std::max(di.maxf, tile_frags(r.len, paired) * tile_frags(c.len, paired));
      di.g0 = (int)gi;
      while (gi < sc->groups.size() && sc->groups[gi].dst == d) {
        const Group& g = sc->groups[gi];
        di.cost[g.fused] += (int64_t)g.tcount * group_seg_cost(g, di.maxf);   // heaviest tile of the block
        di.nseg[g.fused] += g.tcount;
        ++gi;
      }
      di.g1 = (int)gi;
      for (int pass = 0; pass < 2; ++pass) total_cost[pass] += di.cost[pass] * (int64_t)(di.rt.size() * di.ct.size());
    }
  }
  // Fewer waves for smaller problems: the partials a launch writes (and reduce_kernel reads back) grow with the number of
  // units, not with the problem - 48 waves are ~0.9 GB whatever D is, 0.14 ms of a 2.7 ms apply at D = 2048 (measured
  // there: 12-24 waves 25.3-25.7 TFLOPS, 48 waves 24.7; at D = 4096 48 waves are still best).
  const int auto_waves = (int)std::max<int64_t>(8, std::min<int64_t>(48, total_cost[0] / 3400000));
  const int waves = opt.p2_waves > 0 ? opt.p2_waves : auto_waves;
  // 4 resident CTAs per SM, ~48 waves: small units keep the tail of the launch short and the operand segments of a
  // (block, K-chunk) bundle L2-resident while its tiles pass over them.  Measured A/B/A/B on B200, 32 -> 48 waves:
  // cyp 31.6 -> 32.0 TFLOPS, stress 32.2 -> 32.5, femoco 31.7 -> 32.0, small unchanged (p2 -2 %, reduce +0.035 ms);
  // 64 waves gain nothing more (the ordered reduce grows as fast as p2 shrinks).
  const int64_t slots = std::max<int64_t>(1, (int64_t)std::max(n_sm, 1) * 4 * waves / nvec);   // every unit exists once per vector
  const int64_t min_target = opt.p2_min_unit_dmma > 0 ? opt.p2_min_unit_dmma : 3072;   // DMMA per unit at least (~20 us of a CTA; D = 1024: 17.9 -> 18.9 TFLOPS against 1536)
  sc->tuning[1] = waves;
  sc->tuning[2] = min_target;
  const int64_t target_of[2] = {std::max<int64_t>(min_target, total_cost[0] / slots),
                                std::max<int64_t>(min_target, total_cost[1] / slots)};

  sc->runs.clear(); sc->p2.clear(); sc->pf.clear();
  std::vector<int> unit_bundle[2];         // (block, split) bundle of each unit, per pass
  std::vector<int64_t> bundle_cost[2];     // heaviest tile of the bundle, in DMMA count
  int64_t issued_p2 = 0;
  for (int d = 0; d < nB; ++d) {
    PsiBlk& D = sc->blocks[d];
    D.ldo = sector_up(D.cols);
    D.part_off = ws;
    D.nsplit = 0;
    const auto& rt = dsts[d].rt;
    const auto& ct = dsts[d].ct;
    const int maxf = dsts[d].maxf;
    int realised = 0;
    for (int pass = 0; pass < 2; ++pass) {
      if (dsts[d].nseg[pass] == 0) continue;
      std::vector<P2Unit>& units = pass ? sc->pf : sc->p2;
      const int64_t target = target_of[pass];
      int64_t nsplit = (dsts[d].cost[pass] + target - 1) / target;
      nsplit = std::max<int64_t>(1, std::min<int64_t>(nsplit, dsts[d].nseg[pass]));
      // cut the seg sequence of this pass at cumulative cost boundaries
      int64_t cum = 0;
      int gi = dsts[d].g0;
      int ti = 0;                                    // position inside group gi
      auto skip_other = [&]() { while (gi < dsts[d].g1 && sc->groups[gi].fused != pass) { ++gi; ti = 0; } };
      skip_other();
      for (int64_t sp = 0; sp < nsplit; ++sp) {
        const int64_t want = dsts[d].cost[pass] * (sp + 1) / nsplit;
        int run0 = (int)sc->runs.size();
        int64_t chunk_ksteps = 0;
        while (gi < dsts[d].g1 && (cum < want || sp == nsplit - 1)) {
          const Group& g = sc->groups[gi];
          const int64_t per = group_seg_cost(g, maxf);
          int take;
          if (sp == nsplit - 1) take = g.tcount - ti;
          else take = (int)std::min<int64_t>(g.tcount - ti, std::max<int64_t>(1, (want - cum + per - 1) / per));
          if (take > 0) {
            // a run has one storage layout of its operator blocks: split [ti, ti + take) at every layout change
            // (adjoint-pair sharing gives one boundary per group; arbitrary flags may alternate)
            for (int s0 = ti; s0 < ti + take;) {
              const int32_t tr = sc->segs[g.seg0 + s0].p2_trans;
              int s1 = s0 + 1;
              while (s1 < ti + take && sc->segs[g.seg0 + s1].p2_trans == tr) ++s1;
              Run r{g.seg0 + s0, g.seg0 + s1, g.N1, g.ldw, g.order, g.rows, g.seg0, g.ws_map, g.ws_off, tr, 0, 0, 0, g.N1p, 0};
              if (g.fused) { r.K1 = g.K1; r.y1_map = g.y1_map; r.ldy1 = g.ldy1; r.y1_off = g.y1_off; }
              sc->runs.push_back(r);
              s0 = s1;
            }
            cum += per * take;
            chunk_ksteps += (int64_t)((g.N1 + 3) / 4) * take;
            ti += take;
          }
          if (ti >= g.tcount) { ++gi; ti = 0; skip_other(); }
        }
        int run1 = (int)sc->runs.size();
        if (run1 == run0) continue;                  // empty chunk (rounding): skip
        int64_t bundle_max = 0;
        for (auto& r : rt)
          for (auto& c : ct) {
            P2Unit u{};
            u.run_begin = run0; u.run_end = run1;
            u.i0 = r.start; u.rows_valid = r.len; u.j0 = c.start; u.cols_valid = c.len;
            u.ldo = D.ldo;
            const int fm = tile_frags(r.len, paired), fn = tile_frags(c.len, paired);
            u.grid = pass ? 2 : best_grid(fm, fn, nullptr, paired);       // fused CTAs: 2x2 warps, <= 4x4 fragments each
            for (int v = 0; v < nvec; ++v) {              // the vectors of a tile are adjacent: they read the same operator tile
              u.vec = v;
              u.out_off = ws + ((int64_t)realised * nvec + v) * D.rows * D.ldo + (int64_t)r.start * D.ldo + c.start;
              units.push_back(u);
              unit_bundle[pass].push_back((int)bundle_cost[pass].size());
            }
            int64_t dmma = (int64_t)fm * fn * chunk_ksteps;
            int64_t cost = 0;                         // this tile's cost over the chunk's runs, stage floor included
            for (int ri = run0; ri < run1; ++ri) {
              const Run& rr = sc->runs[ri];
              Group gg{};
              gg.N1 = rr.K;
              int64_t per = seg_cost(gg, (int64_t)fm * fn);
              if (pass) {                             // first GEMM of the fused segment on its own tile
                const int64_t fa = (int64_t)(rr.order == 1 ? fm : fn) * frags(rr.K);
                gg.K1 = rr.K1;
                per += fused_extra(gg, fa);
                dmma += fa * ((rr.K1 + 3) / 4) * (rr.seg_end - rr.seg_begin);
              }
              cost += (int64_t)(rr.seg_end - rr.seg_begin) * per;
            }
            int heavy = 0;
            best_grid(fm, fn, &heavy, paired);
            sc->critical_flops += (int64_t)NCONS_WARPS * heavy * chunk_ksteps * 512;
            bundle_max = std::max(bundle_max, cost);
            issued_p2 += dmma * 512;
          }
        bundle_cost[pass].push_back(bundle_max);
        ++realised;
      }
    }
    D.nsplit = realised;
    ws = align_up(ws + (int64_t)realised * nvec * D.rows * D.ldo, 16);
  }
  // LPT order over (block, split) bundles: the tiles of one bundle read the same operand segments, so they stay
  // adjacent in launch order (co-resident CTAs -> the second reader hits L2); bundles go heaviest tile first.
  for (int pass = 0; pass < 2; ++pass) {
    std::vector<P2Unit>& units = pass ? sc->pf : sc->p2;
    std::vector<int> idx(units.size());
    std::iota(idx.begin(), idx.end(), 0);
    const auto& ub = unit_bundle[pass];
    const auto& bc = bundle_cost[pass];
    std::stable_sort(idx.begin(), idx.end(), [&](int a, int b) {
      if (bc[ub[a]] != bc[ub[b]]) return bc[ub[a]] > bc[ub[b]];
      return ub[a] < ub[b];
    });
    std::vector<P2Unit> sorted(units.size());
    for (size_t i = 0; i < idx.size(); ++i) sorted[i] = units[idx[i]];
    units.swap(sorted);
  }
  sc->issued_flops = sc->issued_flops_p1 + issued_p2;
  sc->ws_len = std::max<int64_t>(ws, 16);
  return HPSI_OK;
}

}  // namespace hpsi
