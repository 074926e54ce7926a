// Fused kernel for narrow groups (north_star: "the intermediate block kept in shared memory or registers between the two
// GEMMs"; DESIGN.md section 4 says when it pays).  One CTA = one P2Unit of Schedule::pf: an output tile of a destination
// block and a K-chunk of that block's FUSED segments (tasks).  Per segment
//   phase A: C1[i, j] = coef * sum_k XA[i,k] YA[j,k]   (first GEMM; order 1: XA = A_t rows of the tile, YA = padded psi^T
//            block; order 2: XA = B_t rows of the tile's columns, YA = padded psi block; all N1 <= 64 columns at once),
//            accumulated in registers and written to a shared-memory operand buffer in the swizzled K-tile layout the
//            fragment loads expect - the intermediate never leaves the SM;
//   phase B: out_tile += sum_k X[i,k] Y[j,k] with that buffer as X (order 1, Y = B_t) or as Y (order 2, X = A_t),
//            accumulated in registers over all segments of the unit and written once as a split-K partial.
// Same producer / consumer structure, stage ring and tile layout as kernels.cu; 2x2 warp grid, <= 4x4 fragments per warp
// for both accumulator sets (fragment counts are run-time here: predicated DMMA), 2 CTAs per SM.
#include "kernels_common.cuh"

namespace hpsi {

constexpr int TBUF_BYTES = (TILE / KT) * OP_BYTES;                // the intermediate as <= 4 K-tiles of 64 rows x 128 bytes
constexpr int SMEM_FUSED = 1024 + NSTAGE * STAGE_BYTES + TBUF_BYTES + 2 * NSTAGE * 8;

__device__ __forceinline__ void consumer_barrier() { asm volatile("bar.sync 1, %0;\n" ::"n"(NCONS * 32) : "memory"); }

// nk4 k-steps of up to 4x4 fragments, fragment counts known at run time (warp-uniform predicates)
__device__ __forceinline__ void mma_stage_rt(const double* px, const double* py, const LaneOffsets& lo, double (&acc)[4][4][2],
                                             int mi, int nj, int nk4) {
#pragma unroll
  for (int ks = 0; ks < 4; ++ks) {
    if (ks < nk4) {
      double a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) a[i] = (i < mi) ? px[lo.k[ks] + i * 128] : 0.0;
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = (j < nj) ? py[lo.k[ks] + j * 128] : 0.0;
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j)
          if (i < mi && j < nj) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
    }
  }
}

template <bool TMA>
__global__ void __launch_bounds__(NTHREADS, 2) pf_kernel(DevSchedule d) {
  pdl_wait();
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const P2Unit u = d.pf[blockIdx.x];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const SmemLayout sm(smem_raw);
  // the intermediate's buffer sits between the stages and the barriers of the common layout: shift the barriers
  const uint32_t tbuf_s = sm.base + NSTAGE * STAGE_BYTES;
  double* tbuf = const_cast<double*>(sm.gen) + NSTAGE * (STAGE_BYTES / 8);
  auto full_bar = [&](int s) { return tbuf_s + TBUF_BYTES + s * 8; };
  auto empty_bar = [&](int s) { return tbuf_s + TBUF_BYTES + (NSTAGE + s) * 8; };
  if (tid == 0) {
    for (int s = 0; s < NSTAGE; ++s) { mbar_init(full_bar(s), TMA ? 1 : 32); mbar_init(empty_bar(s), NCONS); }
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  for (int e = tid; e < TBUF_BYTES / 8; e += NTHREADS) tbuf[e] = 0.0;     // no NaN may sit in rows / columns nobody writes
  __syncthreads();

  if (wid == NCONS) {
    // ---------------- producer warp: per segment the stages of phase A (two boxes), then of phase B (one box)
    Ring ring{0, 1};
    for (int ri = u.run_begin; ri < u.run_end; ++ri) {
      const Run r = d.runs[ri];
      const int rowA = (r.order == 1) ? u.i0 : u.j0;               // first row of the phase-A operator tile
      const int rowsA = (r.order == 1) ? u.rows_valid : u.cols_valid;
      const int rowB = (r.order == 1) ? u.j0 : u.i0;               // first row of the phase-B operator tile
      const int rowsB = (r.order == 1) ? u.cols_valid : u.rows_valid;
      const int nta = (r.K1 + KT - 1) / KT, ntb = (r.K + KT - 1) / KT;
      const unsigned char* ymap = d.maps + (int64_t)r.y1_map * TMAP_BYTES;
      const double* ybase = d.ws + r.y1_off;
      const double* arenaA = (r.order == 1) ? d.a : d.b;
      const double* arenaB = (r.order == 1) ? d.b : d.a;
      for (int si = r.seg_begin; si < r.seg_end; ++si) {
        const Seg* sg = d.segs + si;
        if (TMA && lane == 0 && si + 2 < r.seg_end) {              // descriptors of the segment after next
          tma_prefetch_desc(d.maps + (int64_t)sg[2].p1_map * TMAP_BYTES);
          tma_prefetch_desc(d.maps + (int64_t)sg[2].p2_map * TMAP_BYTES);
        }
        for (int kt = 0; kt < nta + ntb; ++kt) {
          mbar_wait(empty_bar(ring.stage), ring.phase);
          const uint32_t sx = sm.stage(ring.stage), sy = sx + X_BOXES * OP_BYTES, full = full_bar(ring.stage);
          if (kt < nta) {                                          // phase A: X = operator rows, Y = psi-side block
            if (TMA) {
              if (lane == 0) {
                mbar_arrive_expect_tx(full, 2 * OP_BYTES);
                tma_load_2d(sx, d.maps + (int64_t)sg->p1_map * TMAP_BYTES, kt * KT, rowA, full);
                tma_load_2d(sy, ymap, kt * KT, 0, full);
              }
            } else {
              ldgsts_tile(sx, arenaA + sg->p1_off + (int64_t)rowA * sg->p1_ld, sg->p1_ld, rowsA, kt * KT, r.K1, lane);
              ldgsts_tile(sy, ybase, r.ldy1, r.K, kt * KT, r.K1, lane);
              cp_async_mbar_arrive(full);
            }
          } else {                                                 // phase B: the operator tile into the slot the buffer does not replace
            const int kb = (kt - nta) * KT;
            const uint32_t dst = (r.order == 1) ? sy : sx;
            if (TMA) {
              if (lane == 0) {
                mbar_arrive_expect_tx(full, OP_BYTES);
                tma_load_2d(dst, d.maps + (int64_t)sg->p2_map * TMAP_BYTES, kb, rowB, full);
              }
            } else {
              ldgsts_tile(dst, arenaB + sg->p2_off + (int64_t)rowB * sg->p2_ld, sg->p2_ld, rowsB, kb, r.K, lane);
              cp_async_mbar_arrive(full);
            }
          }
          ring.advance();
        }
      }
    }
    if (!TMA) cp_async_wait_all();
    return;
  }

  // ------------------ consumer warps (2x2 grid)
  const int warp = (wid + quadrant_rotation(blockIdx.x)) % NCONS;
  const WarpTile wB(2, warp, u.rows_valid, u.cols_valid);          // this warp's part of the output tile
  const LaneOffsets lo(lane);
  const int pg = frag_perm(lane >> 2), pc = frag_perm(2 * (lane & 3));
  double acc2[4][4][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc2[i][j][0] = acc2[i][j][1] = 0.0;
  Ring ring{0, 0};
  for (int ri = u.run_begin; ri < u.run_end; ++ri) {
    const Run r = d.runs[ri];
    const int rowsA = (r.order == 1) ? u.rows_valid : u.cols_valid;
    const WarpTile wA(2, warp, rowsA, r.K);                        // this warp's part of the intermediate (rowsA x N1)
    const int nta = (r.K1 + KT - 1) / KT, ntb = (r.K + KT - 1) / KT;
    const int lastA = ((r.K1 - (nta - 1) * KT) + 3) >> 2, lastB = ((r.K - (ntb - 1) * KT) + 3) >> 2;
    for (int si = r.seg_begin; si < r.seg_end; ++si) {
      const double coef = d.segs[si].coef;
      double acc1[4][4][2];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc1[i][j][0] = acc1[i][j][1] = 0.0;
      for (int kt = 0; kt < nta; ++kt) {                           // phase A
        mbar_wait(full_bar(ring.stage), ring.phase);
        const double* st = sm.stage_ptr(ring.stage);
        mma_stage_rt(st + wA.wr0 * 16, st + X_BOXES * OP_BYTES / 8 + wA.wc0 * 16, lo, acc1, wA.mi, wA.nj, kt == nta - 1 ? lastA : 4);
        __syncwarp();
        if (lane == 0) mbar_arrive(empty_bar(ring.stage));
        ring.advance();
      }
      consumer_barrier();                                          // everybody is done reading the previous segment's buffer
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j)
          if (i < wA.mi && j < wA.nj) {
            const int row = wA.wr0 + 8 * i + pg;
#pragma unroll
            for (int e = 0; e < 2; ++e) {
              const int col = wA.wc0 + 8 * j + pc + 2 * e, c = col & 15;
              tbuf[(col >> 4) * (OP_BYTES / 8) + row * 16 + ((((c >> 1) ^ (row & 7)) << 1) | (c & 1))] = acc1[i][j][e] * coef;
            }
          }
      consumer_barrier();                                          // the intermediate is complete
      for (int kt = 0; kt < ntb; ++kt) {                           // phase B
        mbar_wait(full_bar(ring.stage), ring.phase);
        const double* st = sm.stage_ptr(ring.stage);
        const double* tk = tbuf + kt * (OP_BYTES / 8);
        const double* px = (r.order == 1) ? tk + wB.wr0 * 16 : st + wB.wr0 * 16;
        const double* py = (r.order == 1) ? st + X_BOXES * OP_BYTES / 8 + wB.wc0 * 16 : tk + wB.wc0 * 16;
        mma_stage_rt(px, py, lo, acc2, wB.mi, wB.nj, kt == ntb - 1 ? lastB : 4);
        __syncwarp();
        if (lane == 0) mbar_arrive(empty_bar(ring.stage));
        ring.advance();
      }
    }
  }
  double* dst = d.ws + u.out_off;
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j)
      if (i < wB.mi && j < wB.nj) {
        const int row = wB.wr0 + 8 * i + pg, col = wB.wc0 + 8 * j + pc;
        if (row < u.rows_valid) {
          if (col < u.cols_valid) dst[(int64_t)row * u.ldo + col] = acc2[i][j][0];
          if (col + 2 < u.cols_valid) dst[(int64_t)row * u.ldo + col + 2] = acc2[i][j][1];
        }
      }
}

cudaError_t kernels_fused_init() {
  cudaError_t e;
  if ((e = cudaFuncSetAttribute(pf_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_FUSED))) return e;
  return cudaFuncSetAttribute(pf_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_FUSED);
}

void launch_pf(const DevSchedule& d, bool tma, cudaStream_t st) {
  if (d.n_pf == 0) return;
  if (tma) launch_dependent(pf_kernel<true>, dim3(d.n_pf), dim3(NTHREADS), SMEM_FUSED, st, d);
  else launch_dependent(pf_kernel<false>, dim3(d.n_pf), dim3(NTHREADS), SMEM_FUSED, st, d);
}

}  // namespace hpsi
