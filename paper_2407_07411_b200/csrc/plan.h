// Internal schedule format shared by the host planner, the host schedule interpreter and the kernels.
// Flat POD tables only: the same bytes are uploaded to the device and walked by hpsi_debug_interpret.
//
// Vocabulary:
//   task   = (term t, A block l<-l', B block r<-r') with (l',r') and (l,r) both psi blocks          (8(a)-2)
//   group  = all tasks with the same (source psi block, destination psi block); they share the dims
//            (m,k,n',n), hence the order choice, and are STACKED along one GEMM dimension            (8(a)-4)
//   seg    = one task seen as a K-segment of the second GEMM / a row-segment of the first GEMM
//   P1     = first GEMM  (order 1: T_t = c_t A_t psi ; order 2: U_t^T = c_t B_t psi^T), stacked over the group's terms
//   P2     = second GEMM (order 1: out += T_t B_t^T ; order 2: out += A_t U_t), K runs over all segs of all groups
//            that write one destination block; split-K partials + ordered reduce, no atomics on data.
// Every GEMM is "NT": C[i,j] = sum_k X[i,k] * Y[j,k] with both operands K-contiguous.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/hpsi.h"

namespace hpsi {

constexpr int TILE = 64;      // CTA tile columns (max) and rows of one TMA box, 8 fragments of 8
constexpr int TILE_M = 64;    // CTA tile rows (max)
constexpr int KT = 16;        // K extent of one staged tile (4 DMMA k-steps)
constexpr int NCONS_WARPS = 4;   // consumer (DMMA) warps per CTA (3 CTAs / SM)

enum BaseSel : int32_t { BASE_A = 0, BASE_B = 1, BASE_WS = 2 };
// How the consumer warps of a CTA cover its tile: P1Unit / P2Unit `grid` = number of warp COLUMNS gn (a power of two
// dividing NCONS_WARPS); the warps form a (NCONS_WARPS / gn) x gn grid.

struct Seg {                  // one task, in schedule order (by destination, source, term)
  int64_t p1_off;             // operator block used by P1 (order 1: A_t, order 2: B_t), doubles into its arena
  int64_t p2_off;             // operator block used by P2 (order 1: B_t, order 2: A_t)
  int32_t p1_ld, p2_ld;       // leading dimensions of those blocks
  int32_t p1_map, p2_map;     // tensor-map ids of those blocks (TMA staging)
  double coef;                // per-task coefficient (initialised to c_t; reading A4)
  int32_t p1_trans, p2_trans; // 1: that block is stored transposed (hpsi_terms_t a_transposed / b_transposed)
};

struct Group {
  int32_t order;              // 1 or 2
  int32_t tcount;             // tasks (terms) in the group
  int32_t seg0;               // first Seg
  int32_t rows;               // rows of one task's intermediate (order 1: m, order 2: n)
  int32_t K1;                 // P1 contraction length (order 1: k, order 2: n')
  int32_t N1;                 // P1 columns = P2 segment length (order 1: n', order 2: k)
  int32_t ldw;                // leading dimension of the intermediate (N1 rounded up to a multiple of 4)
  int32_t ldy1;               // leading dimension of the P1 Y operand (padded psi^T or psi block)
  int64_t y1_off;             // its offset in the workspace
  int64_t ws_off;             // start of the stacked intermediate  [(tcount*rows) x ldw]; task t starts at row t*rows
  int32_t y1_map;             // tensor map of the P1 Y operand
  int32_t ws_map;             // tensor map of the stacked intermediate
  int32_t src, dst;           // psi block indices
  int32_t fused;              // 1: narrow group, both GEMMs run in one CTA (kernels_fused.cu): no P1 unit, no workspace intermediate
  int32_t N1p;                // batched plans (nvec > 1): columns one vector occupies in the intermediate (N1 rounded up to 16,
                              // pad columns stay zero), vector v at column v * N1p; single-vector plans: N1
};

struct P1Unit {               // one CTA of the first-GEMM kernel: one tile position, a range of the group's terms
  int32_t group;
  int32_t t0, t1;             // terms [t0, t1) of the group, processed one after the other (pipeline never drains)
  int32_t i0, rows_valid;     // row tile inside one task's intermediate
  int32_t j0, cols_valid;     // column tile
  int32_t grid;               // warp columns gn
  int32_t xtrans;             // 1: the operator blocks of these terms are stored transposed (K-major X operand)
  int32_t vec;                // batched plans: which of the nvec vectors this unit works on
};

struct Run {                  // consecutive segs of one group inside one P2 unit's K range
  int32_t seg_begin, seg_end;
  int32_t K;                  // segment length (group.N1)
  int32_t ldw;                // ld of the intermediate operand
  int32_t order;
  int32_t rows;               // rows of one task's intermediate (group.rows)
  int32_t seg0;               // group.seg0 (seg - seg0 = task index inside the stacked intermediate)
  int32_t ws_map;             // group.ws_map
  int64_t ws_off;             // group.ws_off
  int32_t trans;              // 1: the operator blocks of these segs are stored transposed (K-major operand)
  int32_t K1;                 // fused runs only: contraction length of the first GEMM (group.K1)
  int32_t y1_map, ldy1;       // fused runs only: the first GEMM's shared operand (padded psi^T / psi block), group.y1_map / ldy1
  int32_t Kp;                 // group.N1p: column stride between the vectors of a batched intermediate
  int64_t y1_off;             // fused runs only: group.y1_off
};

struct P2Unit {               // one CTA of the second-GEMM kernel
  int32_t run_begin, run_end;
  int32_t i0, rows_valid, j0, cols_valid;
  int64_t out_off;            // partial buffer offset of element (i0, j0) of this split's m x ldp tile
  int32_t ldo;
  int32_t grid;               // warp columns gn
  int32_t vec;                // batched plans: which of the nvec vectors this unit works on
  int32_t pad;
};

// A 2-D row-major matrix the TMA unit reads: rows x cols doubles as STORED, leading dimension ld, `off` doubles into
// `base`.  Encoded (api.cu) as a CUtensorMap with box {box_cols columns, box_rows rows}, 128-byte swizzle, zero fill
// out of bounds.  K-contiguous operand ("N" layout): rows = the operand's rows, cols = K, box {KT, TILE}.
// Block stored transposed ("T" layout): rows = K, cols = the operand's rows, box {8, KT}, 64-byte swizzle.
struct MapSpec {
  int64_t off;
  int32_t base;               // BaseSel
  int32_t rows, cols, ld;
  int32_t box_rows, box_cols;
};

struct PsiBlk {               // one psi block and its padded copies
  int64_t off;                // in psi / out (dense rows x cols)
  int64_t p_off;              // padded copy   rows x ldp   in workspace
  int64_t t_off;              // padded transpose cols x ldt in workspace
  int32_t rows, cols, ldp, ldt;
  int64_t part_off;           // split-K partials: nsplit x nvec x (rows x ldo), vector fastest
  int64_t p_vstride, t_vstride;   // batched plans: doubles between the padded copies (transposes) of consecutive vectors
  int32_t nsplit, ldo;
  int32_t left, right;
  int32_t diag0, diag1;       // range in the diagonal-task table
  int32_t p_map, t_map;       // tensor maps of the padded copy / padded transpose
};

struct ElemCta {              // one CTA of the element-wise kernels (prep, reduce, diag): 256 consecutive elements of one psi block
  int32_t blk, e0;
};

struct DiagTask {             // sector-diagonal task (for diag(H))
  int64_t a_off, b_off;
  int32_t a_ld, b_ld;
  double coef;
  int32_t seg;                // the task (index into segs) this entry belongs to
  int32_t pad;
};

struct Schedule {
  std::vector<PsiBlk> blocks;
  std::vector<Seg> segs;
  std::vector<Group> groups;
  std::vector<P1Unit> p1;
  std::vector<Run> runs;
  std::vector<P2Unit> p2;
  std::vector<P2Unit> pf;             // units of the fused kernel (same descriptor; their runs are fused runs)
  std::vector<DiagTask> diag;
  std::vector<ElemCta> elem;          // psi elements in granules of 256 per block: no CTA of an element-wise launch is idle
  std::vector<MapSpec> maps;          // tensor maps the TMA kernels use (only filled / valid when aligned16)
  std::vector<hpsi_task_t> tasks;     // schedule order, for hpsi_query
  int64_t psi_len = 0;
  int64_t ws_len = 0;                 // doubles
  int64_t useful_flops = 0, useful_flops_p1 = 0, issued_flops = 0, issued_flops_p1 = 0, operator_bytes = 0, intermediate_bytes = 0;
  int64_t critical_flops = 0;         // 4 warps x the heaviest warp's DMMA flops, summed over units (imbalance included)
  int64_t n_order1 = 0;
  int32_t max_block_elems = 0;
  bool aligned16 = true;              // descriptors allow the 16-byte staging path (arena base checked at bind)
  bool paired = false;                // some block is stored transposed: the GEMMs run the mixed-layout kernels (kernels_paired.cu)
  int64_t tuning[3] = {0, 0, 0};      // realised schedule knobs: P1 K-tiles per unit, P2 waves, P2 minimum DMMA per unit
  int32_t n_terms_planned = 0;        // terms of this plan's shard (all terms without a shard)
  int32_t nvec = 1;                   // vectors one hpsi_apply_multi works on (hpsi_plan_options_t.n_vectors)
};

// What hpsi_plan_ex adds to hpsi_plan (include/hpsi.h hpsi_plan_options_t): a term shard and the schedule knobs.
struct PlanOptions {
  const int32_t* shard_of_term = nullptr;   // [n_terms] or null (= every term)
  int32_t shard_index = 0;
  int32_t p1_stages_per_unit = 0;           // 0 = automatic
  int32_t p2_waves = 0;
  int32_t p2_min_unit_dmma = 0;
  int32_t n_vectors = 0;                    // 0 / 1: single-vector plan
};

// Host planner.  Returns HPSI_OK or an error code with `err` filled.
int build_schedule(const hpsi_sectors_t* s, const hpsi_terms_t* t, uint32_t flags, int n_sm, const PlanOptions& opt,
                   Schedule* out, std::string* err);
// Useful flops (reading A18) of every term: flops[t] = sum over the term's tasks of min(f1, f2).  Descriptors only.
int term_useful_flops(const hpsi_sectors_t* s, const hpsi_terms_t* t, std::vector<int64_t>* flops, std::string* err);

// Tile split of one dimension (planner.cpp): rows up to TILE_M, columns up to TILE, sizes in units of two fragments.
struct Tile1D { int start, len; };
std::vector<Tile1D> split_dim(int64_t n, int max_frags, int unit);
std::vector<Tile1D> split_rows(int64_t n);
std::vector<Tile1D> split_cols(int64_t n);

// Host interpreter of the schedule (tests only; naive loops).
void interpret_schedule(const Schedule& sc, const double* a, const double* b, const double* psi, double* out, int nvec = 1);   // vectors psi_len apart

inline int even_up(int x) { return x + (x & 1); }
// Plan-owned matrices (padded psi, intermediates, partials) start every row on a 32-byte L2 sector, so that a staged
// 128-byte row segment is exactly four sectors (measured: 16-byte-aligned rows cost 1.4x the sectors).
inline int sector_up(int x) { return (x + 3) & ~3; }
inline int frags(int x) { return (x + 7) / 8; }
// fragments a tile dimension of x rows occupies (plans with transposed blocks use 8-row fragments too, kernels_paired.cu)
inline int tile_frags(int x, bool /*paired*/) { return (x + 7) / 8; }
// Heaviest warp (in fragments) when a tile of fm x fn fragments is covered by a gm x gn grid of warps, and the grid
// that minimises it among those whose warp tile has a compiled instantiation (<=4x4, <=8x2, <=2x8 fragments);
// ties go to the squarest grid (fewest shared-memory reads per DMMA).
inline int heaviest_warp(int fm, int fn, int gm, int gn) { return ((fm + gm - 1) / gm) * ((fn + gn - 1) / gn); }
inline bool warp_tile_ok(int mi, int nj) { return (mi <= 4 && nj <= 4) || (mi <= 8 && nj <= 2) || (mi <= 2 && nj <= 8); }
inline int32_t best_grid(int fm, int fn, int* heaviest = nullptr, bool /*paired*/ = false) {
  const int order[4] = {2, 4, 1, NCONS_WARPS};   // squarest first
  int best = 1 << 30;
  int32_t g = 2;
  for (int gn : order) {
    if (gn > NCONS_WARPS || NCONS_WARPS % gn) continue;
    const int gm = NCONS_WARPS / gn;
    if (!warp_tile_ok((fm + gm - 1) / gm, (fn + gn - 1) / gn)) continue;
    const int h = heaviest_warp(fm, fn, gm, gn);
    if (h < best) { best = h; g = gn; }
  }
  if (heaviest) *heaviest = best;
  return g;
}

}  // namespace hpsi
