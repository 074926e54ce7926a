// sm_100a kernels of hpsi_apply: prep (padded psi, psi^T), P1 (first GEMM, per tile position over a range of terms),
// P2 (segmented-K second GEMM with split-K partials), reduce (ordered sum of partials), diag.
// See kernels.cuh / plan.h for the vocabulary.
//
// GEMM CTA = 1 producer warp + NCONS consumer warps (warp-specialised, mbarrier ring of NSTAGE stages).  Default:
// NCONS = 4 on a <=64x64 tile, 3 CTAs per SM; HPSI_BIG_CTA=1 compiles 8 consumer warps on a <=128x64 tile, 2 CTAs per SM
// (measured slower on B200: 27.7 vs 31.9 TFLOPS on the cyp config).
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
#include "kernels.cuh"

namespace hpsi {

// ----------------------------------------------------------------------------------------------- PTX helpers
__device__ __forceinline__ void cp_async_chunk8(uint32_t dst, const void* src, int bytes) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(dst), "l"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }

__device__ __forceinline__ void mbar_init(uint32_t bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.shared::cta.b64 st, [%0];\n}\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n}\n" ::"r"(bar), "r"(bytes)
               : "memory");
}
// arrive on `bar` once all cp.async issued so far by this thread have landed (does not change the pending count)
__device__ __forceinline__ void cp_async_mbar_arrive(uint32_t bar) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n"
      : "=r"(ok)
      : "r"(bar), "r"(parity)
      : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) {}
}
// TMA tile load: box of the tensor map at column c0 (K index), row c1 -> shared memory, completes on `bar`
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const void* tmap, int c0, int c1, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];\n" ::"r"(dst),
      "l"(tmap), "r"(c0), "r"(c1), "r"(bar)
      : "memory");
}

// D(8x8) += A(8x4,row) * B(4x8,col): lane L, g=L>>2, q=L&3 holds a=A[g][q], b=B[q][g], c0,c1=C[g][2q],C[g][2q+1].
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

// row (or column) of a fragment that lane group / accumulator index x in 0..7 maps to
__device__ __forceinline__ int frag_perm(int x) { return ((x & 3) << 1) | (x >> 2); }

// ------------------------------------------------------------------------------------------------- MMA core
// Balanced split of f fragments over `parts` warps: part p gets ceil or floor of f / parts, heavier parts first.
__device__ __forceinline__ void split_frags(int f, int parts, int p, int& first, int& count) {
  const int base = f / parts, rem = f - base * parts;
  count = base + (p < rem ? 1 : 0);
  first = p * base + (p < rem ? p : rem);
}
// The consumer warps cover the tile as a (NCONS / gn) x gn grid (gn = the unit's `grid`, chosen by the planner so that
// the heaviest warp is as light as possible); a warp owns at most 16 fragments: <=4x4, <=8x2 or <=2x8.
struct WarpTile {
  int wr0, wc0;    // first row / col of the warp inside the CTA tile (multiples of 8)
  int mi, nj;      // fragments owned
  __device__ __forceinline__ WarpTile(int gn, int warp, int rows_valid, int cols_valid) {
    const int gm = NCONS / gn;
    int f0;
    split_frags((rows_valid + 7) >> 3, gm, warp / gn, f0, mi);
    wr0 = f0 * 8;
    split_frags((cols_valid + 7) >> 3, gn, warp % gn, f0, nj);
    wc0 = f0 * 8;
  }
};

// Per-lane element offsets (in doubles, inside an operand tile) of the k-steps 0..3 of a fragment whose first row is
// row 0: row perm(g), column 4*ks + q, swizzled.  Fragment i of a warp adds (w0 + 8 i) * 16.
struct LaneOffsets {
  int k[4];
  __device__ __forceinline__ LaneOffsets(int lane) {
    const int g = lane >> 2, q = lane & 3, pg = frag_perm(g);
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) k[ks] = pg * 16 + (((2 * ks + (q >> 1)) ^ pg) << 1) + (q & 1);
  }
};

template <int MI, int NJ>
__device__ __forceinline__ void mma_step(const double (&a)[MI], const double (&b)[NJ], double (&acc)[MI][NJ][2]) {
#pragma unroll
  for (int i = 0; i < MI; ++i)
#pragma unroll
    for (int j = 0; j < NJ; ++j) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
}
template <int MI, int NJ>
__device__ __forceinline__ void load_frags(const double* px, const double* py, int off, double (&a)[MI], double (&b)[NJ]) {
#pragma unroll
  for (int i = 0; i < MI; ++i) a[i] = px[off + i * 128];
#pragma unroll
  for (int j = 0; j < NJ; ++j) b[j] = py[off + j * 128];
}
// One staged K-tile for a warp owning MI x NJ fragments (compile-time, so no predicated DMMA and no WARPSYNC):
// nk4 k-steps of MI*NJ DMMA.8x8x4; the fragments of step ks+1 are fetched while step ks issues.
// px / py = the warp's first row of the X / Y tile of the stage.
template <int MI, int NJ>
__device__ __forceinline__ void mma_stage(const double* px, const double* py, const LaneOffsets& lo,
                                          double (&acc)[MI][NJ][2], int nk4) {
  double a0[MI], b0[NJ], a1[MI], b1[NJ];
  load_frags<MI, NJ>(px, py, lo.k[0], a0, b0);
  if (nk4 == 4) {                       // the common case: straight-line, no predication, no WARPSYNC
    load_frags<MI, NJ>(px, py, lo.k[1], a1, b1);
    mma_step<MI, NJ>(a0, b0, acc);
    load_frags<MI, NJ>(px, py, lo.k[2], a0, b0);
    mma_step<MI, NJ>(a1, b1, acc);
    load_frags<MI, NJ>(px, py, lo.k[3], a1, b1);
    mma_step<MI, NJ>(a0, b0, acc);
    mma_step<MI, NJ>(a1, b1, acc);
  } else {                              // ragged K tail of a segment (1..3 k-steps)
    mma_step<MI, NJ>(a0, b0, acc);
    if (nk4 > 1) { load_frags<MI, NJ>(px, py, lo.k[1], a0, b0); mma_step<MI, NJ>(a0, b0, acc); }
    if (nk4 > 2) { load_frags<MI, NJ>(px, py, lo.k[2], a0, b0); mma_step<MI, NJ>(a0, b0, acc); }
  }
}

template <int MI, int NJ>
__device__ __forceinline__ void zero_acc(double (&acc)[MI][NJ][2]) {
#pragma unroll
  for (int i = 0; i < MI; ++i)
#pragma unroll
    for (int j = 0; j < NJ; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
}

// Store the warp's accumulators: element (row, col) of the CTA tile goes to dst[row*ld + col], scaled by sc.
// acc[i][j][e] holds tile row wr0 + 8i + perm(g) and tile column wc0 + 8j + perm(2q + e)  (perm(2q+1) = perm(2q) + 2).
template <int MI, int NJ>
__device__ __forceinline__ void store_tile(double* dst, int ld, int rows_valid, int cols_valid,
                                           const double (&acc)[MI][NJ][2], const WarpTile& w, int lane, double sc) {
  const int pg = frag_perm(lane >> 2), pc = frag_perm(2 * (lane & 3));
#pragma unroll
  for (int i = 0; i < MI; ++i) {
    const int row = w.wr0 + 8 * i + pg;
    if (row >= rows_valid) continue;
    double* drow = dst + (int64_t)row * ld;
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
      const int col = w.wc0 + 8 * j + pc;
      if (col < cols_valid) drow[col] = acc[i][j][0] * sc;
      if (col + 2 < cols_valid) drow[col + 2] = acc[i][j][1] * sc;
    }
  }
}

// Which tile quadrant consumer warp 0 takes.  Consumer warp w sits on SM sub-partition w, and with odd fragment counts
// the quadrants carry unequal DMMA counts (e.g. 16/12/12/9), so co-resident CTAs must not all put their heavy
// quadrant on the same sub-partition.  CTAs are dealt to SMs round-robin (148 = 0 mod 4), hence a hash, not bid & 3.
__device__ __forceinline__ int quadrant_rotation(unsigned bid) { return (int)((bid * 2654435761u) >> 28); }

// Shared-memory carve-up: NSTAGE stages of [X tile | Y tile] (1024-byte aligned), then the barriers.
struct SmemLayout {
  uint32_t base;                                   // shared-window address of stage 0 (1024-byte aligned)
  const double* gen;                               // generic pointer to the same byte
  __device__ __forceinline__ SmemLayout(const void* raw) {
    const uint32_t r = (uint32_t)__cvta_generic_to_shared(raw);
    base = (r + 1023u) & ~1023u;
    gen = reinterpret_cast<const double*>(static_cast<const char*>(raw) + (base - r));
  }
  __device__ __forceinline__ uint32_t stage(int s) const { return base + s * STAGE_BYTES; }
  __device__ __forceinline__ const double* stage_ptr(int s) const { return gen + s * (STAGE_BYTES / 8); }
  __device__ __forceinline__ uint32_t full(int s) const { return base + NSTAGE * STAGE_BYTES + s * 8; }
  __device__ __forceinline__ uint32_t empty(int s) const { return base + NSTAGE * STAGE_BYTES + (NSTAGE + s) * 8; }
};
// TMA: the full barrier takes the producer's arrive.expect_tx plus the bytes; LDGSTS: one deferred arrive per lane.
template <bool TMA>
__device__ __forceinline__ void init_barriers(const SmemLayout& sm, int tid) {
  if (tid == 0) {
    for (int s = 0; s < NSTAGE; ++s) { mbar_init(sm.full(s), TMA ? 1 : 32); mbar_init(sm.empty(s), NCONS); }
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();
}

// position in the stage ring
struct Ring {
  int stage;
  uint32_t phase;
  __device__ __forceinline__ void advance() { if (++stage == NSTAGE) { stage = 0; phase ^= 1; } }
};

// ------------------------------------------------------------------------------------------ LDGSTS staging
// Fallback for matrices with 8-byte aligned rows: the producer warp copies a rows_valid x (K - kappa, at most 16)
// piece with 8-byte cp.async into the swizzled layout; everything else of the 64 x 16 tile is zero-filled.
// Lane handles column (lane & 15) of rows (lane >> 4) + 2 p.
__device__ __forceinline__ void ldgsts_tile(uint32_t s_op, const double* rows, int64_t ld, int rows_valid, int kappa, int K,
                                            int lane) {
  const int kc = lane & 15, r0 = lane >> 4;
  const bool kvalid = kappa + kc < K;
#pragma unroll 8
  for (int p = 0; p < TILE / 2; ++p) {
    const int r = r0 + 2 * p;
    const bool ok = kvalid && r < rows_valid;
    const double* src = ok ? rows + r * ld + kappa + kc : rows;
    const uint32_t dst = s_op + r * 128 + ((((kc >> 1) ^ (r & 7)) << 4) | ((kc & 1) << 3));
    cp_async_chunk8(dst, src, ok ? 8 : 0);
  }
}

// ------------------------------------------------------------------------------------------------ P1 kernel
// One CTA = one P1Unit: for each term t of the unit, T_t[i0.., j0..] = coef_t * sum_k X_t[i,k] Y[j,k] with
// X_t = the term's operator block (order 1: A_t, order 2: B_t) and Y = padded psi^T (order 1) or padded psi
// (order 2) block of the source.  The stage ring runs across the terms.
template <int MI, int NJ>
__device__ __forceinline__ void p1_consume(const DevSchedule& d, const P1Unit& u, const Group& g, const SmemLayout& sm,
                                           const WarpTile& w, int lane) {
  double acc[MI][NJ][2];
  const LaneOffsets lo(lane);
  const int ntiles = (g.K1 + KT - 1) / KT;
  const int last_nk4 = ((g.K1 - (ntiles - 1) * KT) + 3) >> 2;
  Ring ring{0, 0};
  for (int t = u.t0; t < u.t1; ++t) {
    const double coef = d.segs[g.seg0 + t].coef;            // issued before the K loop, needed after it
    zero_acc<MI, NJ>(acc);
    for (int kt = 0; kt < ntiles; ++kt) {
      mbar_wait(sm.full(ring.stage), ring.phase);
      if (d.debug != 2) {
        const double* st = sm.stage_ptr(ring.stage);
        mma_stage<MI, NJ>(st + w.wr0 * 16, st + X_BOXES * OP_BYTES / 8 + w.wc0 * 16, lo, acc, kt == ntiles - 1 ? last_nk4 : 4);
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(sm.empty(ring.stage));
      ring.advance();
    }
    double* dst = d.ws + g.ws_off + ((int64_t)t * g.rows + u.i0) * g.ldw + u.j0;
    store_tile<MI, NJ>(dst, g.ldw, u.rows_valid, u.cols_valid, acc, w, lane, coef);
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

template <bool TMA>
__global__ void __maxnreg__(HPSI_BIG_CTA ? 112 : 136) p1_kernel(DevSchedule d) {
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
    const unsigned char* ymap = d.maps + (int64_t)g.y1_map * TMAP_BYTES;
    const double* ybase = d.ws + g.y1_off + (int64_t)u.j0 * g.ldy1;
    const double* xarena = (g.order == 1) ? d.a : d.b;
    const int xboxes = (u.rows_valid + TILE - 1) / TILE;          // 64-row boxes of the X tile that hold valid rows
    for (int t = u.t0; t < u.t1; ++t) {
      const Seg* sg = d.segs + g.seg0 + t;
      const unsigned char* xmap = nullptr;
      const double* xbase = nullptr;
      int64_t xld = 0;
      if (TMA) xmap = d.maps + (int64_t)sg->p1_map * TMAP_BYTES;
      else { xld = sg->p1_ld; xbase = xarena + sg->p1_off + (int64_t)u.i0 * xld; }
      for (int kt = 0; kt < ntiles; ++kt) {
        mbar_wait(sm.empty(ring.stage), ring.phase);
        const uint32_t sx = sm.stage(ring.stage), sy = sx + X_BOXES * OP_BYTES, full = sm.full(ring.stage);
        if (TMA) {
          if (lane == 0) {
            mbar_arrive_expect_tx(full, d.debug == 1 ? 0 : (xboxes + 1) * OP_BYTES);
            if (d.debug != 1) {
              for (int bx = 0; bx < xboxes; ++bx) tma_load_2d(sx + bx * OP_BYTES, xmap, kt * KT, u.i0 + bx * TILE, full);
              tma_load_2d(sy, ymap, kt * KT, u.j0, full);
            }
          }
        } else {
          if (d.debug != 1) {
            for (int bx = 0; bx < xboxes; ++bx)
              ldgsts_tile(sx + bx * OP_BYTES, xbase + bx * TILE * xld, xld, u.rows_valid - bx * TILE, kt * KT, g.K1, lane);
            ldgsts_tile(sy, ybase, g.ldy1, u.cols_valid, kt * KT, g.K1, lane);
          }
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
#define HPSI_CASE(MI, NJ) case MI * 9 + NJ: p1_consume<MI, NJ>(d, u, g, sm, w, lane); break;
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
    if (d.debug != 2) {
      const double* st = sm.stage_ptr(ring.stage);
      mma_stage<MI, NJ>(st + w.wr0 * 16, st + X_BOXES * OP_BYTES / 8 + w.wc0 * 16, lo, acc, it.nk4());
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(sm.empty(ring.stage));
    ring.advance();
  }
  store_tile<MI, NJ>(d.ws + u.out_off, u.ldo, u.rows_valid, u.cols_valid, acc, w, lane, 1.0);
}

template <bool TMA>
__global__ void __maxnreg__(HPSI_BIG_CTA ? 112 : 136) p2_kernel(DevSchedule d) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const P2Unit u = d.p2[blockIdx.x];
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
    const double *xbase = nullptr, *ybase = nullptr;           // LDGSTS: first rows and leading dimensions
    int64_t xld = 0, yld = 0;
    auto open_seg = [&]() {
      const Run r = d.runs[it.run];
      const Seg* sg = d.segs + it.seg;
      const int trow = (it.seg - r.seg0) * r.rows;             // first row of the task inside the stacked intermediate
      if (TMA) {
        const unsigned char* opmap = d.maps + (int64_t)sg->p2_map * TMAP_BYTES;
        const unsigned char* wsmap = d.maps + (int64_t)r.ws_map * TMAP_BYTES;
        if (r.order == 1) { xmap = wsmap; xrow = trow + u.i0; ymap = opmap; yrow = u.j0; }
        else              { xmap = opmap; xrow = u.i0; ymap = wsmap; yrow = trow + u.j0; }
      } else {
        const double* wsrows = d.ws + r.ws_off + (int64_t)trow * r.ldw;
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
          mbar_arrive_expect_tx(full, d.debug == 1 ? 0 : (xboxes + 1) * OP_BYTES);
          if (d.debug != 1) {
            for (int bx = 0; bx < xboxes; ++bx) tma_load_2d(sx + bx * OP_BYTES, xmap, it.kappa, xrow + bx * TILE, full);
            tma_load_2d(sy, ymap, it.kappa, yrow, full);
          }
        }
      } else {
        if (d.debug != 1) {
          for (int bx = 0; bx < xboxes; ++bx)
            ldgsts_tile(sx + bx * OP_BYTES, xbase + bx * TILE * xld, xld, u.rows_valid - bx * TILE, it.kappa, it.K, lane);
          ldgsts_tile(sy, ybase, yld, u.cols_valid, it.kappa, it.K, lane);
        }
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
// prep: psi block (rows x cols, dense) -> padded copy (rows x ldp) and padded transpose (cols x ldt) in the workspace.
__global__ void prep_kernel(DevSchedule d, const double* __restrict__ psi) {
  const PsiBlk B = d.blocks[blockIdx.y];
  const int n = B.rows * B.cols;
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
    const int x = e / B.cols, y = e - x * B.cols;
    const double v = psi[B.off + e];
    d.ws[B.p_off + (int64_t)x * B.ldp + y] = v;
    d.ws[B.t_off + (int64_t)y * B.ldt + x] = v;
  }
}

// reduce: out block = sum of its split-K partials in split order (fixed order -> bitwise reproducible);
// a block nobody writes (nsplit == 0) becomes zeros (step 5: overwrite semantics).
__global__ void reduce_kernel(DevSchedule d, double* __restrict__ out) {
  const PsiBlk B = d.blocks[blockIdx.y];
  const int n = B.rows * B.cols;
  const int64_t stride = (int64_t)B.rows * B.ldo;
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
    const int x = e / B.cols, y = e - x * B.cols;
    const double* p = d.ws + B.part_off + (int64_t)x * B.ldo + y;
    double s = 0.0;
    for (int sp = 0; sp < B.nsplit; ++sp) s += p[sp * stride];
    out[B.off + e] = s;
  }
}

// diag(H): diag[l][x,y] = sum over sector-diagonal tasks of c_t A[x,x] B[y,y]   (reading A21)
__global__ void diag_kernel(DevSchedule d, double* __restrict__ diag) {
  const PsiBlk B = d.blocks[blockIdx.y];
  const int n = B.rows * B.cols;
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
    const int x = e / B.cols, y = e - x * B.cols;
    double s = 0.0;
    for (int i = B.diag0; i < B.diag1; ++i) {
      const DiagTask t = d.diag[i];
      s += t.coef * d.a[t.a_off + (int64_t)x * t.a_ld + x] * d.b[t.b_off + (int64_t)y * t.b_ld + y];
    }
    diag[B.off + e] = s;
  }
}

// -------------------------------------------------------------------------------------------------- launchers
cudaError_t kernels_init() {
  cudaError_t e;
  if ((e = cudaFuncSetAttribute(p1_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES))) return e;
  if ((e = cudaFuncSetAttribute(p1_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES))) return e;
  if ((e = cudaFuncSetAttribute(p2_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES))) return e;
  if ((e = cudaFuncSetAttribute(p2_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES))) return e;
  return cudaSuccess;
}

static dim3 elem_grid(const DevSchedule& d) {
  int gx = (d.max_block_elems + 255) / 256;
  if (gx < 1) gx = 1;
  if (gx > 1024) gx = 1024;
  return dim3(gx, d.n_blocks);
}

void launch_prep(const DevSchedule& d, const double* psi, cudaStream_t st) {
  if (d.n_blocks > 0) prep_kernel<<<elem_grid(d), 256, 0, st>>>(d, psi);
}
void launch_p1(const DevSchedule& d, bool tma, cudaStream_t st) {
  if (d.n_p1 == 0) return;
  if (tma) p1_kernel<true><<<d.n_p1, NTHREADS, SMEM_BYTES, st>>>(d);
  else p1_kernel<false><<<d.n_p1, NTHREADS, SMEM_BYTES, st>>>(d);
}
void launch_p2(const DevSchedule& d, bool tma, cudaStream_t st) {
  if (d.n_p2 == 0) return;
  if (tma) p2_kernel<true><<<d.n_p2, NTHREADS, SMEM_BYTES, st>>>(d);
  else p2_kernel<false><<<d.n_p2, NTHREADS, SMEM_BYTES, st>>>(d);
}
void launch_reduce(const DevSchedule& d, double* out, cudaStream_t st) {
  if (d.n_blocks > 0) reduce_kernel<<<elem_grid(d), 256, 0, st>>>(d, out);
}
void launch_diag(const DevSchedule& d, double* diag, cudaStream_t st) {
  if (d.n_blocks > 0) diag_kernel<<<elem_grid(d), 256, 0, st>>>(d, diag);
}

}  // namespace hpsi
