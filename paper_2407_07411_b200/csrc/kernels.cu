// sm_100a kernels of hpsi_apply: prep (padded psi, psi^T), P1 (first GEMM, per tile position over a range of terms),
// P2 (segmented-K second GEMM with split-K partials), reduce (ordered sum of partials), diag.
// See kernels.cuh / plan.h for the vocabulary.
//
// GEMM CTA = 1 producer warp + NCONS = 4 consumer warps on a <=64x64 tile (warp-specialised, mbarrier ring of NSTAGE
// stages), 3 CTAs per SM.  (8 consumer warps on a <=128x64 tile at 2 CTAs per SM measured slower: 27.7 vs 31.9 TFLOPS.)
//   producer : one elected lane issues two TMA tile loads per stage (cp.async.bulk.tensor.2d: a 64-row x 16-column
//              box of the X operand and one of the Y operand, 128-byte swizzle, rows / columns past the matrix edge
//              zero-filled by the hardware) that complete on the stage's "full" mbarrier (complete_tx::bytes).
//              Measured on B200 for this access pattern: TMA boxes feed 6.1-6.9 TB/s from HBM and 12-13.9 TB/s from L2,
//              16-byte LDGSTS 4.8 / 6.4 TB/s.  Matrices whose rows are not 16-byte aligned take the LDGSTS variant
//              (8-byte cp.async with zero fill into the same swizzled layout).
//   consumers: a (NCONS / gn) x gn grid of warps, each <= 16 fragments of DMMA.8x8x4 with register accumulators; a warp waits only on the
//              "full" barrier of its next stage and releases the stage on its "empty" barrier - no CTA-wide barrier
//              in the main loop.
//
// Shared-memory tile layout (what the TMA unit writes with CU_TENSOR_MAP_SWIZZLE_128B): row r of a tile is 128
// bytes (16 doubles); its 16-byte chunk c sits at chunk position c ^ (r & 7).  A fragment (8 rows x 4 k) is read
// conflict-free when the 4 rows of each half-warp have distinct (r & 7) >> 1, so lane group g of a fragment reads row
// perm(g) = (0,2,4,6,1,3,5,7)[g] of the fragment's 8 rows; the accumulator rows / columns are permuted accordingly
// when the tile is stored.
#include <algorithm>

#include "kernels_common.cuh"

namespace hpsi {

// ------------------------------------------------------------------------------------------------ P1 kernel
// One CTA = one P1Unit: for each term t of the unit, T_t[i0.., j0..] = coef_t * sum_k X_t[i,k] Y[j,k] with
// X_t = the term's operator block (order 1: A_t, order 2: B_t) and Y = padded psi^T (order 1) or padded psi
// (order 2) block of the source.  The stage ring runs across the terms.
// ROT (operator update, rotate.cu): the tile of term t is stored transposed at rot_dst + Seg.p2_off with ld Seg.p2_ld.
template <int MI, int NJ, bool ROT>
__device__ __forceinline__ void p1_consume(const DevSchedule& d, const P1Unit& u, const Group& g, const SmemLayout& sm,
                                           const WarpTile& w, int lane) {
  double acc[MI][NJ][2];
  const LaneOffsets lo(lane);
  const int ntiles = (g.K1 + KT - 1) / KT;
  const int last_nk4 = ((g.K1 - (ntiles - 1) * KT) + 3) >> 2;
  Ring ring{0, 0};
  for (int t = u.t0; t < u.t1; ++t) {
    const double coef = ROT ? 1.0 : d.segs[g.seg0 + t].coef;   // issued before the K loop, needed after it
    zero_acc<MI, NJ>(acc);
    for (int kt = 0; kt < ntiles; ++kt) {
      mbar_wait(sm.full(ring.stage), ring.phase);
      const double* st = sm.stage_ptr(ring.stage);
      mma_stage<MI, NJ>(st + w.wr0 * 16, st + X_BOXES * OP_BYTES / 8 + w.wc0 * 16, lo, acc, kt == ntiles - 1 ? last_nk4 : 4);
      __syncwarp();
      if (lane == 0) mbar_arrive(sm.empty(ring.stage));
      ring.advance();
    }
    if (ROT && g.N1p > 0) {
      // operator update, second launch (rotate.cu): "term" t is the slab of 64 rows [64 t, 64 t + 64) of the group's
      // STACKED first-GEMM results (N1p rows per block, the first g.ldw of them real); row R of the stack belongs to
      // block R / N1p and goes, transposed, to that block's A' at Seg.p2_off / p2_ld
      const int pg = frag_perm(lane >> 2), pc = frag_perm(2 * (lane & 3));
#pragma unroll
      for (int i = 0; i < MI; ++i) {
        const int R = t * TILE + w.wr0 + 8 * i + pg;
        if (R >= g.rows) continue;
        const int blk = R / g.N1p, a = R - blk * g.N1p;
        if (a >= g.ldw) continue;
        const Seg* sg = d.segs + g.seg0 + blk;
        double* dst = d.rot_dst + sg->p2_off + a;
#pragma unroll
        for (int j = 0; j < NJ; ++j) {
          const int col = w.wc0 + 8 * j + pc;
          if (col < u.cols_valid) dst[(int64_t)(u.j0 + col) * sg->p2_ld] = acc[i][j][0];
          if (col + 2 < u.cols_valid) dst[(int64_t)(u.j0 + col + 2) * sg->p2_ld] = acc[i][j][1];
        }
      }
    } else if (ROT) {
      const Seg* sg = d.segs + g.seg0 + t;
      store_tile_t<MI, NJ>(d.rot_dst + sg->p2_off + (int64_t)u.j0 * sg->p2_ld + u.i0, sg->p2_ld, u.rows_valid, u.cols_valid, acc, w, lane);
    } else {
      double* dst = d.ws + g.ws_off + ((int64_t)t * g.rows + u.i0) * g.ldw + u.vec * g.N1p + u.j0;
      store_tile<MI, NJ>(dst, g.ldw, u.rows_valid, u.cols_valid, acc, w, lane, coef);
    }
  }
}
// a consumer warp without fragments (tile narrower than the warp grid) only hands the stages back
__device__ __forceinline__ void idle_consume(const SmemLayout& sm, int nstages, int lane) {
  Ring ring{0, 0};
  for (int i = 0; i < nstages; ++i) {
    mbar_wait(sm.full(ring.stage), ring.phase);
    if (lane == 0) mbar_arrive(sm.empty(ring.stage));
    ring.advance();
  }
}

// Dispatch to the instantiation for the warp's (mi, nj): <=4x4 (2x2 grid), <=8x2 (1x4 grid), <=2x8 (4x1 grid).
#define HPSI_DISPATCH_FRAGS(CALL)                                                                               \
  switch (w.mi * 9 + w.nj) {                                                                                    \
    CALL(1, 1) CALL(1, 2) CALL(1, 3) CALL(1, 4) CALL(2, 1) CALL(2, 2) CALL(2, 3) CALL(2, 4)                     \
    CALL(3, 1) CALL(3, 2) CALL(3, 3) CALL(3, 4) CALL(4, 1) CALL(4, 2) CALL(4, 3) CALL(4, 4)                     \
    CALL(5, 1) CALL(5, 2) CALL(6, 1) CALL(6, 2) CALL(7, 1) CALL(7, 2) CALL(8, 1) CALL(8, 2)                     \
    CALL(1, 5) CALL(2, 5) CALL(1, 6) CALL(2, 6) CALL(1, 7) CALL(2, 7) CALL(1, 8) CALL(2, 8)                     \
    default: __trap();                                                                                          \
  }

template <bool TMA, bool ROT>
__global__ void __maxnreg__(136) p1_kernel(DevSchedule d) {
  pdl_wait();
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const P1Unit u = d.p1[blockIdx.x];
  if (!ROT && u.vec >= d.nvec_active) return;            // batched plan applied to fewer vectors than it was laid out for
  const Group g = d.groups[u.group];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const SmemLayout sm(smem_raw);
  init_barriers<TMA>(sm, tid);
  const int ntiles = (g.K1 + KT - 1) / KT;
  const int yrow0 = u.vec * g.N1 + u.j0;                 // the Y operand of vector v starts at row v * N1 of the stacked copies

  if (wid == NCONS) {
    // ---------------- producer warp
    Ring ring{0, 1};
    const unsigned char* ymap = d.maps + (int64_t)g.y1_map * TMAP_BYTES;
    const double* ybase = d.ws + g.y1_off + (int64_t)yrow0 * g.ldy1;
    const double* xarena = (g.order == 1) ? d.a : d.b;
    const int xboxes = (u.rows_valid + TILE - 1) / TILE;          // 64-row boxes of the X tile that hold valid rows
    const bool stacked = ROT && g.N1p > 0;                         // "terms" are 64-row slabs of one stacked matrix (see p1_consume)
    for (int t = u.t0; t < u.t1; ++t) {
      const Seg* sg = d.segs + g.seg0 + (stacked ? 0 : t);
      const unsigned char* xmap = nullptr;
      const double* xbase = nullptr;
      int64_t xld = 0;
      const int xrow0 = stacked ? t * TILE : u.i0;
      const int xrows = stacked ? min(TILE, g.rows - t * TILE) : u.rows_valid;
      if (TMA) {
        xmap = d.maps + (int64_t)sg->p1_map * TMAP_BYTES;
        if (!stacked && lane == 0 && t + 2 < u.t1) tma_prefetch_desc(d.maps + (int64_t)sg[2].p1_map * TMAP_BYTES);   // descriptor of the term after next
      } else { xld = sg->p1_ld; xbase = xarena + sg->p1_off + (int64_t)xrow0 * xld; }
      for (int kt = 0; kt < ntiles; ++kt) {
        mbar_wait(sm.empty(ring.stage), ring.phase);
        const uint32_t sx = sm.stage(ring.stage), sy = sx + X_BOXES * OP_BYTES, full = sm.full(ring.stage);
        if (TMA) {
          if (lane == 0) {
            mbar_arrive_expect_tx(full, (xboxes + 1) * OP_BYTES);
            for (int bx = 0; bx < xboxes; ++bx) tma_load_2d(sx + bx * OP_BYTES, xmap, kt * KT, xrow0 + bx * TILE, full);
            tma_load_2d(sy, ymap, kt * KT, yrow0, full);
          }
        } else {
          for (int bx = 0; bx < xboxes; ++bx)
            ldgsts_tile(sx + bx * OP_BYTES, xbase + bx * TILE * xld, xld, xrows - bx * TILE, kt * KT, g.K1, lane);
          ldgsts_tile(sy, ybase, g.ldy1, u.cols_valid, kt * KT, g.K1, lane);
          cp_async_mbar_arrive(full);
        }
        ring.advance();
      }
    }
    if (!TMA) cp_async_wait_all();
    return;
  }

  // ------------------ consumer warps
  const int warp = (wid + quadrant_rotation(blockIdx.x)) % NCONS;
  const WarpTile w(u.grid, warp, u.rows_valid, u.cols_valid);
  if (w.mi == 0 || w.nj == 0) { idle_consume(sm, ntiles * (u.t1 - u.t0), lane); return; }
#define HPSI_CASE(MI, NJ) case MI * 9 + NJ: p1_consume<MI, NJ, ROT>(d, u, g, sm, w, lane); break;
  HPSI_DISPATCH_FRAGS(HPSI_CASE)
#undef HPSI_CASE
}

// ------------------------------------------------------------------------------------------------ P2 kernel
// One CTA = one P2Unit: partial[i0.., j0..] = sum over the unit's runs, segs and k of X[i,k] Y[j,k]
// (order 1: X = T_t from the workspace, Y = B_t; order 2: X = A_t, Y = U_t^T from the workspace).
struct KIter {                 // walks (run, seg, kappa) in K-tile steps
  const Run* runs;
  int run, run_end, seg, seg_end, K, kappa;
  bool valid;
  __device__ __forceinline__ void open_run() {
    seg = runs[run].seg_begin; seg_end = runs[run].seg_end; K = runs[run].K; kappa = 0;
  }
  __device__ __forceinline__ KIter(const Run* runs_, int rb, int re) : runs(runs_), run(rb), run_end(re) {
    valid = rb < re;
    if (valid) open_run();
  }
  // returns true if the segment changed
  __device__ __forceinline__ bool advance() {
    kappa += KT;
    if (kappa < K) return false;
    kappa = 0;
    if (++seg < seg_end) return true;
    if (++run < run_end) { open_run(); return true; }
    valid = false;
    return false;
  }
  __device__ __forceinline__ int nk4() const { int n = (K - kappa + 3) >> 2; return n > 4 ? 4 : n; }
};

template <int MI, int NJ>
__device__ __forceinline__ void p2_consume(const DevSchedule& d, const P2Unit& u, const SmemLayout& sm,
                                           const WarpTile& w, int lane) {
  double acc[MI][NJ][2];
  zero_acc<MI, NJ>(acc);
  const LaneOffsets lo(lane);
  Ring ring{0, 0};
  for (KIter it(d.runs, u.run_begin, u.run_end); it.valid; it.advance()) {
    mbar_wait(sm.full(ring.stage), ring.phase);
    const double* st = sm.stage_ptr(ring.stage);
    mma_stage<MI, NJ>(st + w.wr0 * 16, st + X_BOXES * OP_BYTES / 8 + w.wc0 * 16, lo, acc, it.nk4());
    __syncwarp();
    if (lane == 0) mbar_arrive(sm.empty(ring.stage));
    ring.advance();
  }
  store_tile<MI, NJ>(d.ws + u.out_off, u.ldo, u.rows_valid, u.cols_valid, acc, w, lane, 1.0);
}

template <bool TMA>
__global__ void __maxnreg__(136) p2_kernel(DevSchedule d) {
  pdl_wait();
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const P2Unit u = d.p2[blockIdx.x];
  if (u.vec >= d.nvec_active) return;                    // batched plan applied to fewer vectors than it was laid out for
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const SmemLayout sm(smem_raw);
  init_barriers<TMA>(sm, tid);

  if (wid == NCONS) {
    // ---------------- producer warp
    KIter it(d.runs, u.run_begin, u.run_end);
    Ring ring{0, 1};
    const int xboxes = (u.rows_valid + TILE - 1) / TILE;          // 64-row boxes of the X tile that hold valid rows
    const unsigned char *xmap = nullptr, *ymap = nullptr;      // TMA: tensor maps and first rows of the segment
    int xrow = 0, yrow = 0;
    int xcol = 0, ycol = 0;                                    // batched plans: first column of this unit's vector in the intermediate
    const double *xbase = nullptr, *ybase = nullptr;           // LDGSTS: first rows and leading dimensions
    int64_t xld = 0, yld = 0;
    auto open_seg = [&]() {
      const Run r = d.runs[it.run];
      const Seg* sg = d.segs + it.seg;
      const int trow = (it.seg - r.seg0) * r.rows;             // first row of the task inside the stacked intermediate
      if (TMA) {
        const unsigned char* opmap = d.maps + (int64_t)sg->p2_map * TMAP_BYTES;
        const unsigned char* wsmap = d.maps + (int64_t)r.ws_map * TMAP_BYTES;
        if (lane == 0 && it.seg + 2 < r.seg_end) tma_prefetch_desc(d.maps + (int64_t)sg[2].p2_map * TMAP_BYTES);   // descriptor of the segment after next
        if (r.order == 1) { xmap = wsmap; xrow = trow + u.i0; xcol = u.vec * r.Kp; ymap = opmap; yrow = u.j0; ycol = 0; }
        else              { xmap = opmap; xrow = u.i0; xcol = 0; ymap = wsmap; yrow = trow + u.j0; ycol = u.vec * r.Kp; }
      } else {
        const double* wsrows = d.ws + r.ws_off + (int64_t)trow * r.ldw + u.vec * r.Kp;
        if (r.order == 1) {
          xld = r.ldw; xbase = wsrows + (int64_t)u.i0 * xld;
          yld = sg->p2_ld; ybase = d.b + sg->p2_off + (int64_t)u.j0 * yld;
        } else {
          xld = sg->p2_ld; xbase = d.a + sg->p2_off + (int64_t)u.i0 * xld;
          yld = r.ldw; ybase = wsrows + (int64_t)u.j0 * yld;
        }
      }
    };
    if (it.valid) open_seg();
    while (it.valid) {
      mbar_wait(sm.empty(ring.stage), ring.phase);
      const uint32_t sx = sm.stage(ring.stage), sy = sx + X_BOXES * OP_BYTES, full = sm.full(ring.stage);
      if (TMA) {
        if (lane == 0) {
          mbar_arrive_expect_tx(full, (xboxes + 1) * OP_BYTES);
          for (int bx = 0; bx < xboxes; ++bx) tma_load_2d(sx + bx * OP_BYTES, xmap, xcol + it.kappa, xrow + bx * TILE, full);
          tma_load_2d(sy, ymap, ycol + it.kappa, yrow, full);
        }
      } else {
        for (int bx = 0; bx < xboxes; ++bx)
          ldgsts_tile(sx + bx * OP_BYTES, xbase + bx * TILE * xld, xld, u.rows_valid - bx * TILE, it.kappa, it.K, lane);
        ldgsts_tile(sy, ybase, yld, u.cols_valid, it.kappa, it.K, lane);
        cp_async_mbar_arrive(full);
      }
      if (it.advance()) open_seg();
      ring.advance();
    }
    if (!TMA) cp_async_wait_all();
    return;
  }

  // ------------------ consumer warps
  const int warp = (wid + quadrant_rotation(blockIdx.x)) % NCONS;
  const WarpTile w(u.grid, warp, u.rows_valid, u.cols_valid);
  if (w.mi == 0 || w.nj == 0) {
    int nstages = 0;
    for (KIter it(d.runs, u.run_begin, u.run_end); it.valid; it.advance()) ++nstages;
    idle_consume(sm, nstages, lane);
    return;
  }
#define HPSI_CASE(MI, NJ) case MI * 9 + NJ: p2_consume<MI, NJ>(d, u, sm, w, lane); break;
  HPSI_DISPATCH_FRAGS(HPSI_CASE)
#undef HPSI_CASE
}

// ------------------------------------------------------------------------------- prep / reduce / diag kernels
// Element-wise launches run one CTA per ElemCta granule (256 consecutive elements of one psi block): every CTA has work,
// whatever the spread of block sizes (a (largest block / 256) x n_blocks grid left most CTAs of the small blocks idle:
// reduce 0.030 -> see DESIGN.md on the D = 1024 config).  blockIdx.y = vector of a batched apply.
//
// prep: psi block (rows x cols, dense) -> padded copy (rows x ldp) and padded transpose (cols x ldt) in the workspace.
// With nrm2 given, psi is first divided by sqrt(nrm2[v]) and the normalised vector is also written to `normalized` (the
// eigensolver drivers hand over a new basis vector unnormalised: one launch fewer per iteration).
__global__ void prep_kernel(DevSchedule d, const double* __restrict__ psi, const double* __restrict__ nrm2,
                            double* __restrict__ normalized) {
  pdl_wait();
  const ElemCta c = d.elem[blockIdx.x];
  const PsiBlk B = d.blocks[c.blk];
  const int e = c.e0 + threadIdx.x;
  if (e >= B.rows * B.cols) return;
  const int v_ = blockIdx.y;
  const int x = e / B.cols, y = e - x * B.cols;
  double v = psi[(int64_t)v_ * d.ld_psi + B.off + e];
  if (nrm2) { v *= 1.0 / sqrt(nrm2[v_]); normalized[(int64_t)v_ * d.ld_psi + B.off + e] = v; }
  d.ws[B.p_off + v_ * B.p_vstride + (int64_t)x * B.ldp + y] = v;
  d.ws[B.t_off + v_ * B.t_vstride + (int64_t)y * B.ldt + x] = v;
}

// reduce: out block = sum of its split-K partials in a fixed order -> bitwise reproducible; a block nobody writes
// (nsplit == 0) becomes zeros (step 5: overwrite semantics).  Eight lanes share one element: lane q adds the partials of
// splits [q * per, (q + 1) * per) in order (eight loads in flight), then the eight sums are added in lane order.  (One
// thread per element walked up to ~80 dependent L2 round trips: 0.079 -> 0.040 ms of a 0.59 ms apply at D = 1024.)
// Large vectors are bandwidth-bound and lose with eight rows in flight per warp (cyp 0.115 -> 0.207 ms): they take
// reduce_plain_kernel below; the launcher picks by size.  Partials: split-major, vector-minor.
constexpr int RED_LANES = 8;
__global__ void reduce_kernel(DevSchedule d, double* __restrict__ out, int accumulate) {
  pdl_wait();
  const ElemCta c = d.elem[blockIdx.x >> 3];                   // eight CTAs per granule: 32 elements each (lanes x 8 = 256 threads)
  const PsiBlk B = d.blocks[c.blk];
  const int n = B.rows * B.cols;
  const int64_t stride = (int64_t)d.nvec * B.rows * B.ldo;
  out += (int64_t)blockIdx.y * d.ld_out;
  const double* part = d.ws + B.part_off + (int64_t)blockIdx.y * B.rows * B.ldo;
  const int q = threadIdx.x & (RED_LANES - 1);
  const int per = (B.nsplit + RED_LANES - 1) / RED_LANES;
  const int sp0 = min(q * per, B.nsplit), sp1 = min(sp0 + per, B.nsplit);
  constexpr int EPP = 256 / RED_LANES;                         // elements per CTA
  {                                                            // whole warps stay in for the shuffles
    const int e = c.e0 + (blockIdx.x & 7) * EPP + (threadIdx.x / RED_LANES);
    double s = 0.0;
    if (e < n) {
      const int x = e / B.cols, y = e - x * B.cols;
      const double* p = part + (int64_t)x * B.ldo + y;
      int sp = sp0;
      for (; sp + 8 <= sp1; sp += 8) {
        double v[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) v[i] = __ldg(p + (sp + i) * stride);
#pragma unroll
        for (int i = 0; i < 8; ++i) s += v[i];
      }
      for (; sp < sp1; ++sp) s += __ldg(p + sp * stride);
    }
    // lane 0 of the group collects the eight sums in lane order
    double tot = s;
#pragma unroll
    for (int i = 1; i < RED_LANES; ++i) tot += __shfl_sync(0xffffffffu, s, (threadIdx.x & 31 & ~(RED_LANES - 1)) + i);
    if (q == 0 && e < n) out[B.off + e] = accumulate ? out[B.off + e] + tot : tot;   // hpsi_stream_apply: windows add up in a fixed order
  }
}

// the plain form: one thread per element, rows fully coalesced (large vectors; bandwidth-bound)
__global__ void reduce_plain_kernel(DevSchedule d, double* __restrict__ out, int accumulate) {
  pdl_wait();
  const ElemCta c = d.elem[blockIdx.x];
  const PsiBlk B = d.blocks[c.blk];
  const int e = c.e0 + threadIdx.x;
  if (e >= B.rows * B.cols) return;
  const int64_t stride = (int64_t)d.nvec * B.rows * B.ldo;
  out += (int64_t)blockIdx.y * d.ld_out;
  const int x = e / B.cols, y = e - x * B.cols;
  const double* p = d.ws + B.part_off + (int64_t)blockIdx.y * B.rows * B.ldo + (int64_t)x * B.ldo + y;
  double s = accumulate ? out[B.off + e] : 0.0;             // hpsi_stream_apply: windows of terms add up in a fixed order
  int sp = 0;
  for (; sp + 8 <= B.nsplit; sp += 8) {                     // eight partials in flight, added in split order
    double v[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = __ldg(p + (sp + i) * stride);
#pragma unroll
    for (int i = 0; i < 8; ++i) s += v[i];
  }
  for (; sp < B.nsplit; ++sp) s += __ldg(p + sp * stride);
  out[B.off + e] = s;
}

// diag(H): diag[l][x,y] = sum over sector-diagonal tasks of c_t A[x,x] B[y,y]   (reading A21)
__global__ void diag_kernel(DevSchedule d, double* __restrict__ diag) {
  pdl_wait();
  const ElemCta c = d.elem[blockIdx.x];
  const PsiBlk B = d.blocks[c.blk];
  const int e = c.e0 + threadIdx.x;
  if (e >= B.rows * B.cols) return;
  const int x = e / B.cols, y = e - x * B.cols;
  double s = 0.0;
  for (int i = B.diag0; i < B.diag1; ++i) {
    const DiagTask t = d.diag[i];
    s += t.coef * d.a[t.a_off + (int64_t)x * t.a_ld + x] * d.b[t.b_off + (int64_t)y * t.b_ld + y];
  }
  diag[B.off + e] = s;
}

// out[e] = parts[0][e] + parts[1][e] + ... in that order (term-sharded apply: the ranks' partial H psi, gathered, are added
// in rank order - bitwise the same on every rank and every run, whatever the transport did)
__global__ void sum_shards_kernel(const double* __restrict__ parts, int n_parts, int64_t n, double* __restrict__ out) {
  pdl_wait();
  for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
    double s = parts[e];
    for (int r = 1; r < n_parts; ++r) s += parts[(int64_t)r * n + e];
    out[e] = s;
  }
}
void launch_sum_shards(const double* parts, int n_parts, int64_t n, double* out, cudaStream_t st) {
  if (n <= 0) return;
  const int grid = (int)std::min<int64_t>((n + 255) / 256, 148 * 8);
  sum_shards_kernel<<<grid, 256, 0, st>>>(parts, n_parts, n, out);
}

// -------------------------------------------------------------------------------------------------- launchers
cudaError_t kernels_init() {
  cudaError_t e;
  if ((e = cudaFuncSetAttribute(p1_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES))) return e;
  if ((e = cudaFuncSetAttribute(p1_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES))) return e;
  if ((e = cudaFuncSetAttribute(p1_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES))) return e;
  if ((e = cudaFuncSetAttribute(p1_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES))) return e;
  if ((e = cudaFuncSetAttribute(p2_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES))) return e;
  if ((e = cudaFuncSetAttribute(p2_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES))) return e;
  if ((e = kernels_fused_init())) return e;
  return kernels_paired_init();
}

void launch_prep(const DevSchedule& d, const double* psi, const double* nrm2, double* normalized, cudaStream_t st) {
  if (d.n_elem > 0) launch_dependent(prep_kernel, dim3(dim3(d.n_elem, d.nvec_active)), dim3(256), 0, st, d, psi, nrm2, normalized);
}
void launch_p1(const DevSchedule& d, bool tma, cudaStream_t st) {
  if (d.n_p1 == 0) return;
  if (d.paired) { launch_p1_paired(d, tma, st); return; }
  if (tma) launch_dependent(p1_kernel<true, false>, dim3(d.n_p1), dim3(NTHREADS), SMEM_BYTES, st, d);
  else launch_dependent(p1_kernel<false, false>, dim3(d.n_p1), dim3(NTHREADS), SMEM_BYTES, st, d);
}
void launch_p1_rot(const DevSchedule& d, bool tma, cudaStream_t st) {
  if (d.n_p1 == 0) return;
  if (tma) launch_dependent(p1_kernel<true, true>, dim3(d.n_p1), dim3(NTHREADS), SMEM_BYTES, st, d);
  else launch_dependent(p1_kernel<false, true>, dim3(d.n_p1), dim3(NTHREADS), SMEM_BYTES, st, d);
}
void launch_p2(const DevSchedule& d, bool tma, cudaStream_t st) {
  if (d.n_p2 == 0) return;
  if (d.paired) { launch_p2_paired(d, tma, st); return; }
  if (tma) launch_dependent(p2_kernel<true>, dim3(d.n_p2), dim3(NTHREADS), SMEM_BYTES, st, d);
  else launch_dependent(p2_kernel<false>, dim3(d.n_p2), dim3(NTHREADS), SMEM_BYTES, st, d);
}
void launch_reduce(const DevSchedule& d, double* out, bool accumulate, cudaStream_t st) {
  if (d.n_elem == 0) return;
  const bool small_vec = (int64_t)d.n_elem * 256 <= 500000;     // latency-bound sizes (D <~ 1500)
  if (small_vec) launch_dependent(reduce_kernel, dim3(dim3(d.n_elem * 8, d.nvec_active)), dim3(256), 0, st, d, out, accumulate ? 1 : 0);
  else launch_dependent(reduce_plain_kernel, dim3(dim3(d.n_elem, d.nvec_active)), dim3(256), 0, st, d, out, accumulate ? 1 : 0);
}
void launch_diag(const DevSchedule& d, double* diag, cudaStream_t st) {
  if (d.n_elem > 0) launch_dependent(diag_kernel, dim3(d.n_elem), dim3(256), 0, st, d, diag);
}

}  // namespace hpsi
