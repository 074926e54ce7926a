// GEMM kernels for plans in which some operator block is stored transposed (hpsi_terms_t a_transposed / b_transposed:
// adjoint-pair storage sharing).  Same CTA design as kernels.cu (1 TMA producer warp + 4 DMMA consumer
// warps, mbarrier ring, 8 x 8 fragments, tiles padded to 8); what differs is how a fragment's rows map to tile rows, so
// that one mapping reads BOTH operand layouts without bank conflicts:
//
//   N tile (K-contiguous operand, kernels.cu): one 64-row x 16-k TMA box, 128 bytes per row, 128-byte swizzle: element
//            (row r, k) at  r*128 + (((k >> 1) ^ (r & 7)) << 4) + (k & 1)*8  bytes.
//   T tile (block stored transposed = M-contiguous operand): 8 TMA boxes of 8 rows x 16 k from a tensor map whose inner
//            dimension is the operand's ROW index (64 bytes per k, 64-byte swizzle), box b = rows 8b .. 8b+7 at b*1024:
//            element (row r, k) at  k*64 + ((((r >> 1) ^ (k >> 1)) & 3) << 4) + (r & 1)*8  bytes.
//
// A DMMA fragment is 8 rows x 4 k, lane (g, q) reading (row g, k = 4 ks + q); a 64-bit shared load is served per
// half-warp (g = 0..3 | 4..7).  The N tile is conflict-free iff the 4 rows of a half-warp differ in bits (2,1) of r; the T
// tile iff their (r >> 1, r & 1) pairs and those with r >> 1 flipped in bit 0 are all distinct.  Rows {0,3,4,7 | 1,2,5,6}
// satisfy both, so lane group g reads row perm8(g) = (0,3,4,7,1,2,5,6)[g] of the fragment whatever the layout, and a
// unit whose K range mixes plainly stored and transposed blocks keeps ONE accumulator <-> tile-element mapping.
// (Round 1 used 16-row boxes with the 128-byte swizzle for T tiles, which forced fragments to interleave 16 rows and tiles
// to be padded to 16: issued / useful flops 1.109 instead of 1.059 on cyp, 28.5 vs 31.9 TFLOPS.)
#include "kernels_common.cuh"

namespace hpsi {

// row (0..7) of its fragment that lane group / accumulator index x (0..7) maps to
__device__ __forceinline__ int perm8(int x) { return (int)((0x65217430u >> (4 * x)) & 15u); }

// Per-lane element offsets (doubles, relative to the warp's first fragment of the operand tile) of k-steps 0..3; fragment
// i of the warp adds 128 i in both layouts.  `t` = the operand is an M-contiguous ("T") tile.
struct MixOffsets {
  int x[4], y[4];
  __device__ __forceinline__ static int off(int r, int q, int ks, bool t) {
    if (t) { const int k = 4 * ks + q; return k * 8 + ((((r >> 1) ^ (k >> 1)) & 3) << 1) + (r & 1); }
    return r * 16 + (((2 * ks + (q >> 1)) ^ (r & 7)) << 1) + (q & 1);
  }
  __device__ __forceinline__ void set(int lane, bool xt, bool yt) {
    const int r = perm8(lane >> 2), q = lane & 3;
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) { x[ks] = off(r, q, ks, xt); y[ks] = off(r, q, ks, yt); }
  }
};

template <int MI, int NJ>
__device__ __forceinline__ void load_frags_p(const double* px, const double* py, const MixOffsets& po, int ks,
                                             double (&a)[MI], double (&b)[NJ]) {
#pragma unroll
  for (int i = 0; i < MI; ++i) a[i] = px[po.x[ks] + i * 128];
#pragma unroll
  for (int j = 0; j < NJ; ++j) b[j] = py[po.y[ks] + j * 128];
}
// as mma_stage (kernels.cu): the fragments of k-step ks+1 are fetched while step ks issues
template <int MI, int NJ>
__device__ __forceinline__ void mma_stage_p(const double* px, const double* py, const MixOffsets& po,
                                            double (&acc)[MI][NJ][2], int nk4) {
  double a0[MI], b0[NJ], a1[MI], b1[NJ];
  load_frags_p<MI, NJ>(px, py, po, 0, a0, b0);
  if (nk4 == 4) {
    load_frags_p<MI, NJ>(px, py, po, 1, a1, b1);
    mma_step<MI, NJ>(a0, b0, acc);
    load_frags_p<MI, NJ>(px, py, po, 2, a0, b0);
    mma_step<MI, NJ>(a1, b1, acc);
    load_frags_p<MI, NJ>(px, py, po, 3, a1, b1);
    mma_step<MI, NJ>(a0, b0, acc);
    mma_step<MI, NJ>(a1, b1, acc);
  } else {
    mma_step<MI, NJ>(a0, b0, acc);
    if (nk4 > 1) { load_frags_p<MI, NJ>(px, py, po, 1, a0, b0); mma_step<MI, NJ>(a0, b0, acc); }
    if (nk4 > 2) { load_frags_p<MI, NJ>(px, py, po, 2, a0, b0); mma_step<MI, NJ>(a0, b0, acc); }
  }
}

// acc[i][j][e] holds tile row wr0 + 8 i + perm8(g) and tile column wc0 + 8 j + perm8(2 q + e)
template <int MI, int NJ>
__device__ __forceinline__ void store_tile_p(double* dst, int ld, int rows_valid, int cols_valid,
                                             const double (&acc)[MI][NJ][2], const WarpTile& w, int lane, double sc) {
  const int pg = perm8(lane >> 2), q = lane & 3;
  const int pc0 = perm8(2 * q), pc1 = perm8(2 * q + 1);
#pragma unroll
  for (int i = 0; i < MI; ++i) {
    const int row = w.wr0 + 8 * i + pg;
    if (row >= rows_valid) continue;
    double* drow = dst + (int64_t)row * ld;
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
      const int c0 = w.wc0 + 8 * j + pc0, c1 = w.wc0 + 8 * j + pc1;
      if (c0 < cols_valid) drow[c0] = acc[i][j][0] * sc;
      if (c1 < cols_valid) drow[c1] = acc[i][j][1] * sc;
    }
  }
}

// ---------------------------------------------------------------------------------------------- staging
// LDGSTS fallback for an M-contiguous operand: rows_valid operand rows starting at `first` (= element (row 0, k 0) of
// the window), k-major with leading dimension ld, written in the T-tile layout above.  Lane handles k = lane & 15 of rows
// (lane >> 4) + 2 p.
__device__ __forceinline__ void ldgsts_tile_t(uint32_t s_op, const double* first, int64_t ld, int rows_valid, int kappa,
                                              int K, int lane) {
  const int k = lane & 15, r0 = lane >> 4;
  const bool kvalid = kappa + k < K;
#pragma unroll 8
  for (int p = 0; p < TILE / 2; ++p) {
    const int r = r0 + 2 * p, rr = r & 7;
    const bool ok = kvalid && r < rows_valid;
    const double* src = ok ? first + (int64_t)(kappa + k) * ld + r : first;
    const uint32_t dst = s_op + (r >> 3) * 1024 + k * 64 + (((((rr >> 1) ^ (k >> 1)) & 3) << 4) | ((rr & 1) << 3));
    cp_async_chunk8(dst, src, ok ? 8 : 0);
  }
}

// One operand of a stage.  N: one 64-row x 16-k box (or the 8-byte LDGSTS copy); T: ceil(rows_valid / 8) boxes of
// 16 k x 8 rows.  `row0` = first operand row of the tile inside the matrix; for LDGSTS `ptr` = element (row0, 0).
struct OperandSrc {
  const unsigned char* map;   // TMA
  const double* ptr;          // LDGSTS
  int64_t ld;
  int row0;
  int trans;
};
__device__ __forceinline__ uint32_t operand_bytes(const OperandSrc& o, int rows_valid) {
  return o.trans ? (uint32_t)((rows_valid + 7) >> 3) * 1024u : (uint32_t)OP_BYTES;
}
template <bool TMA>
__device__ __forceinline__ void stage_operand(const OperandSrc& o, uint32_t s_op, int rows_valid, int kappa, int K,
                                              uint32_t full, int lane) {
  if (TMA) {
    if (lane != 0) return;
    if (!o.trans) { tma_load_2d(s_op, o.map, kappa, o.row0, full); return; }
    const int nsub = (rows_valid + 7) >> 3;
    for (int b = 0; b < nsub; ++b) tma_load_2d(s_op + b * 1024, o.map, o.row0 + 8 * b, kappa, full);
  } else {
    if (!o.trans) ldgsts_tile(s_op, o.ptr, o.ld, rows_valid, kappa, K, lane);
    else ldgsts_tile_t(s_op, o.ptr, o.ld, rows_valid, kappa, K, lane);
  }
}
template <bool TMA>
__device__ __forceinline__ void stage_both(const OperandSrc& x, const OperandSrc& y, const SmemLayout& sm, const Ring& ring,
                                           int rows_valid, int cols_valid, int kappa, int K, int lane) {
  const uint32_t sx = sm.stage(ring.stage), sy = sx + X_BOXES * OP_BYTES, full = sm.full(ring.stage);
  if (TMA) {
    if (lane == 0)
      mbar_arrive_expect_tx(full, operand_bytes(x, rows_valid) + operand_bytes(y, cols_valid));
    stage_operand<true>(x, sx, rows_valid, kappa, K, full, lane);
    stage_operand<true>(y, sy, cols_valid, kappa, K, full, lane);
  } else {
    stage_operand<false>(x, sx, rows_valid, kappa, K, full, lane);
    stage_operand<false>(y, sy, cols_valid, kappa, K, full, lane);
    cp_async_mbar_arrive(full);
  }
}

// Dispatch to the instantiation for the warp's (mi, nj): <=4x4 (2x2 grid), <=8x2 (1x4 grid), <=2x8 (4x1 grid), as kernels.cu.
#define HPSI_DISPATCH_PAIRS(CALL)                                                                               \
  switch (w.mi * 9 + w.nj) {                                                                                    \
    CALL(1, 1) CALL(1, 2) CALL(1, 3) CALL(1, 4) CALL(2, 1) CALL(2, 2) CALL(2, 3) CALL(2, 4)                     \
    CALL(3, 1) CALL(3, 2) CALL(3, 3) CALL(3, 4) CALL(4, 1) CALL(4, 2) CALL(4, 3) CALL(4, 4)                     \
    CALL(5, 1) CALL(5, 2) CALL(6, 1) CALL(6, 2) CALL(7, 1) CALL(7, 2) CALL(8, 1) CALL(8, 2)                     \
    CALL(1, 5) CALL(2, 5) CALL(1, 6) CALL(2, 6) CALL(1, 7) CALL(2, 7) CALL(1, 8) CALL(2, 8)                     \
    default: __trap();                                                                                          \
  }

__device__ __forceinline__ void idle_consume_p(const SmemLayout& sm, int nstages, int lane) {
  Ring ring{0, 0};
  for (int i = 0; i < nstages; ++i) {
    mbar_wait(sm.full(ring.stage), ring.phase);
    if (lane == 0) mbar_arrive(sm.empty(ring.stage));
    ring.advance();
  }
}

// ------------------------------------------------------------------------------------------------ P1 kernel
template <int MI, int NJ>
__device__ __forceinline__ void p1p_consume(const DevSchedule& d, const P1Unit& u, const Group& g, const SmemLayout& sm,
                                            const WarpTile& w, int lane) {
  double acc[MI][NJ][2];
  MixOffsets po;
  po.set(lane, u.xtrans != 0, false);
  const int ntiles = (g.K1 + KT - 1) / KT;
  const int last_nk4 = ((g.K1 - (ntiles - 1) * KT) + 3) >> 2;
  Ring ring{0, 0};
  for (int t = u.t0; t < u.t1; ++t) {
    const double coef = d.segs[g.seg0 + t].coef;
    zero_acc<MI, NJ>(acc);
    for (int kt = 0; kt < ntiles; ++kt) {
      mbar_wait(sm.full(ring.stage), ring.phase);
      const double* st = sm.stage_ptr(ring.stage);
      mma_stage_p<MI, NJ>(st + w.wr0 * 16, st + X_BOXES * OP_BYTES / 8 + w.wc0 * 16, po, acc, kt == ntiles - 1 ? last_nk4 : 4);
      __syncwarp();
      if (lane == 0) mbar_arrive(sm.empty(ring.stage));
      ring.advance();
    }
    double* dst = d.ws + g.ws_off + ((int64_t)t * g.rows + u.i0) * g.ldw + u.j0;
    store_tile_p<MI, NJ>(dst, g.ldw, u.rows_valid, u.cols_valid, acc, w, lane, coef);
  }
}

template <bool TMA>
__global__ void __maxnreg__(136) p1p_kernel(DevSchedule d) {
  pdl_wait();
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const P1Unit u = d.p1[blockIdx.x];
  const Group g = d.groups[u.group];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const SmemLayout sm(smem_raw);
  init_barriers<TMA>(sm, tid);
  const int ntiles = (g.K1 + KT - 1) / KT;

  if (wid == NCONS) {
    // ---------------- producer warp
    Ring ring{0, 1};
    const OperandSrc y{d.maps + (int64_t)g.y1_map * TMAP_BYTES, d.ws + g.y1_off + (int64_t)u.j0 * g.ldy1, g.ldy1, u.j0, 0};
    const double* xarena = (g.order == 1) ? d.a : d.b;
    for (int t = u.t0; t < u.t1; ++t) {
      const Seg* sg = d.segs + g.seg0 + t;
      OperandSrc x{d.maps + (int64_t)sg->p1_map * TMAP_BYTES, nullptr, sg->p1_ld, u.i0, u.xtrans};
      if (TMA && lane == 0 && t + 2 < u.t1) tma_prefetch_desc(d.maps + (int64_t)sg[2].p1_map * TMAP_BYTES);   // descriptor of the term after next
      if (!TMA) x.ptr = xarena + sg->p1_off + (u.xtrans ? (int64_t)u.i0 : (int64_t)u.i0 * sg->p1_ld);
      for (int kt = 0; kt < ntiles; ++kt) {
        mbar_wait(sm.empty(ring.stage), ring.phase);
        stage_both<TMA>(x, y, sm, ring, u.rows_valid, u.cols_valid, kt * KT, g.K1, lane);
        ring.advance();
      }
    }
    if (!TMA) cp_async_wait_all();
    return;
  }

  // ------------------ consumer warps
  const int warp = (wid + quadrant_rotation(blockIdx.x)) % NCONS;
  const WarpTile w(u.grid, warp, u.rows_valid, u.cols_valid);
  if (w.mi == 0 || w.nj == 0) { idle_consume_p(sm, ntiles * (u.t1 - u.t0), lane); return; }
#define HPSI_CASE(MI, NJ) case MI * 9 + NJ: p1p_consume<MI, NJ>(d, u, g, sm, w, lane); break;
  HPSI_DISPATCH_PAIRS(HPSI_CASE)
#undef HPSI_CASE
}

// ------------------------------------------------------------------------------------------------ P2 kernel
template <int MI, int NJ>
__device__ __forceinline__ void p2p_consume(const DevSchedule& d, const P2Unit& u, const SmemLayout& sm,
                                            const WarpTile& w, int lane) {
  double acc[MI][NJ][2];
  zero_acc<MI, NJ>(acc);
  MixOffsets po;
  Ring ring{0, 0};
  for (int r = u.run_begin; r < u.run_end; ++r) {            // same (run, seg, k-tile) order as the producer
    const Run run = d.runs[r];
    po.set(lane, run.order == 2 && run.trans, run.order == 1 && run.trans);   // the operator operand may be transposed
    const int K = run.K, nseg = run.seg_end - run.seg_begin;
    const int ntiles = (K + KT - 1) / KT, last_nk4 = ((K - (ntiles - 1) * KT) + 3) >> 2;
    for (int sgi = 0; sgi < nseg; ++sgi)
      for (int kt = 0; kt < ntiles; ++kt) {
        mbar_wait(sm.full(ring.stage), ring.phase);
        const double* st = sm.stage_ptr(ring.stage);
        mma_stage_p<MI, NJ>(st + w.wr0 * 16, st + X_BOXES * OP_BYTES / 8 + w.wc0 * 16, po, acc, kt == ntiles - 1 ? last_nk4 : 4);
        __syncwarp();
        if (lane == 0) mbar_arrive(sm.empty(ring.stage));
        ring.advance();
      }
  }
  store_tile_p<MI, NJ>(d.ws + u.out_off, u.ldo, u.rows_valid, u.cols_valid, acc, w, lane, 1.0);
}

template <bool TMA>
__global__ void __maxnreg__(136) p2p_kernel(DevSchedule d) {
  pdl_wait();
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const P2Unit u = d.p2[blockIdx.x];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const SmemLayout sm(smem_raw);
  init_barriers<TMA>(sm, tid);

  if (wid == NCONS) {
    // ---------------- producer warp
    Ring ring{0, 1};
    for (int r = u.run_begin; r < u.run_end; ++r) {
      const Run run = d.runs[r];
      const unsigned char* wsmap = d.maps + (int64_t)run.ws_map * TMAP_BYTES;
      const int ntiles = (run.K + KT - 1) / KT;
      for (int seg = run.seg_begin; seg < run.seg_end; ++seg) {
        const Seg* sg = d.segs + seg;
        if (TMA && lane == 0 && seg + 2 < run.seg_end) tma_prefetch_desc(d.maps + (int64_t)sg[2].p2_map * TMAP_BYTES);
        const int trow = (seg - run.seg0) * run.rows;          // first row of the task inside the stacked intermediate
        const double* wsrows = d.ws + run.ws_off + (int64_t)trow * run.ldw;
        OperandSrc x, y;
        if (run.order == 1) {                                  // X = T_t (workspace), Y = B_t
          x = OperandSrc{wsmap, wsrows + (int64_t)u.i0 * run.ldw, run.ldw, trow + u.i0, 0};
          y = OperandSrc{d.maps + (int64_t)sg->p2_map * TMAP_BYTES,
                         d.b + sg->p2_off + (run.trans ? (int64_t)u.j0 : (int64_t)u.j0 * sg->p2_ld), sg->p2_ld, u.j0, run.trans};
        } else {                                               // X = A_t, Y = U_t^T (workspace)
          x = OperandSrc{d.maps + (int64_t)sg->p2_map * TMAP_BYTES,
                         d.a + sg->p2_off + (run.trans ? (int64_t)u.i0 : (int64_t)u.i0 * sg->p2_ld), sg->p2_ld, u.i0, run.trans};
          y = OperandSrc{wsmap, wsrows + (int64_t)u.j0 * run.ldw, run.ldw, trow + u.j0, 0};
        }
        for (int kt = 0; kt < ntiles; ++kt) {
          mbar_wait(sm.empty(ring.stage), ring.phase);
          stage_both<TMA>(x, y, sm, ring, u.rows_valid, u.cols_valid, kt * KT, run.K, lane);
          ring.advance();
        }
      }
    }
    if (!TMA) cp_async_wait_all();
    return;
  }

  // ------------------ consumer warps
  const int warp = (wid + quadrant_rotation(blockIdx.x)) % NCONS;
  const WarpTile w(u.grid, warp, u.rows_valid, u.cols_valid);
  if (w.mi == 0 || w.nj == 0) {
    int nstages = 0;
    for (int r = u.run_begin; r < u.run_end; ++r)
      nstages += (d.runs[r].seg_end - d.runs[r].seg_begin) * ((d.runs[r].K + KT - 1) / KT);
    idle_consume_p(sm, nstages, lane);
    return;
  }
#define HPSI_CASE(MI, NJ) case MI * 9 + NJ: p2p_consume<MI, NJ>(d, u, sm, w, lane); break;
  HPSI_DISPATCH_PAIRS(HPSI_CASE)
#undef HPSI_CASE
}

// -------------------------------------------------------------------------------------------------- launchers
cudaError_t kernels_paired_init() {
  cudaError_t e;
  if ((e = cudaFuncSetAttribute(p1p_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES))) return e;
  if ((e = cudaFuncSetAttribute(p1p_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES))) return e;
  if ((e = cudaFuncSetAttribute(p2p_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES))) return e;
  if ((e = cudaFuncSetAttribute(p2p_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES))) return e;
  return cudaSuccess;
}
void launch_p1_paired(const DevSchedule& d, bool tma, cudaStream_t st) {
  if (tma) launch_dependent(p1p_kernel<true>, dim3(d.n_p1), dim3(NTHREADS), SMEM_BYTES, st, d);
  else launch_dependent(p1p_kernel<false>, dim3(d.n_p1), dim3(NTHREADS), SMEM_BYTES, st, d);
}
void launch_p2_paired(const DevSchedule& d, bool tma, cudaStream_t st) {
  if (tma) launch_dependent(p2p_kernel<true>, dim3(d.n_p2), dim3(NTHREADS), SMEM_BYTES, st, d);
  else launch_dependent(p2p_kernel<false>, dim3(d.n_p2), dim3(NTHREADS), SMEM_BYTES, st, d);
}

}  // namespace hpsi
