// sm_100a kernels of hpsi_apply: prep (padded psi, psi^T), P1 (stacked first GEMM), P2 (segmented-K second GEMM
// with split-K partials), reduce (ordered sum of partials), diag.  See kernels.cuh / plan.h for the vocabulary.
//
// GEMM CTA = 1 producer warp + 4 consumer warps (warp-specialised, mbarrier ring of NSTAGE stages):
//   producer : cp.async (LDGSTS, zero-fill for ragged edges) of a 64 x 16 X tile and a 64 x 16 Y tile per stage,
//              completion signalled with cp.async.mbarrier.arrive on the stage's "full" barrier;
//   consumers: 2x2 warps, each <= 4x4 fragments of DMMA.8x8x4 with register accumulators; a warp waits only on the
//              "full" barrier of its next stage and releases the stage on its "empty" barrier - no CTA-wide barrier
//              in the main loop.  Measured on B200: one warp issues a DMMA.8x8x4 at most every ~29 clk while the
//              pipe takes one per 16 clk per SM sub-partition, so >= 2 warps per sub-partition must always be in
//              their DMMA phase; decoupling the warps is what keeps them there.
#include "kernels.cuh"

namespace hpsi {

// ----------------------------------------------------------------------------------------------- PTX helpers
__device__ __forceinline__ void cp_async_chunk16(uint32_t dst, const void* src, int bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(dst), "l"(src), "r"(bytes) : "memory");
}
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

// D(8x8) += A(8x4,row) * B(4x8,col): lane L, g=L>>2, q=L&3 holds a=A[g][q], b=B[q][g], c0,c1=C[g][2q],C[g][2q+1].
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

// ------------------------------------------------------------------------------------------ staging (LDGSTS)
// Stage layout per operand: [k-slab (4)][row (64)][4 doubles]; element (row, kc) at ((kc>>2)*64 + row)*4 + (kc&3).
// A warp's fragment read (row = r0+g, kc = 4*ks+q) is then 32 consecutive doubles: conflict-free.
// CH = doubles per cp.async (2: 16-byte chunks, needs 16-byte aligned rows; 1: 8-byte chunks, any FP64 alignment).
// The producer warp's lane handles chunk column (lane % CPR) of rows (lane / CPR) + p * RPP.
template <int CH>
struct Stager {
  static constexpr int CPR = KT / CH;            // chunks per row
  static constexpr int RPP = 32 / CPR;           // rows per pass of the producer warp
  static constexpr int PASSES = TILE / RPP;
  int r0, kc;
  uint32_t dst0;                                 // byte offset inside an operand's stage
  __device__ __forceinline__ Stager(int lane) {
    const int c = lane % CPR;
    r0 = lane / CPR;
    kc = c * CH;
    dst0 = (uint32_t)((((kc >> 2) * TILE + r0) * 4 + (kc & 3)) * 8);
  }
  // rowptr(p) = pointer to (row r0 + p*RPP, k = 0) in global memory; rows >= rows_valid and k >= K are zero-filled
  template <class RowPtr>
  __device__ __forceinline__ void load(uint32_t s_op, RowPtr rowptr, int rows_valid, const double* safe, int kappa,
                                       int K) const {
    const int kcol = kappa + kc;
    int kvalid = K - kcol;
    kvalid = kvalid < 0 ? 0 : (kvalid > CH ? CH : kvalid);
#pragma unroll
    for (int p = 0; p < PASSES; ++p) {
      const int r = r0 + p * RPP;
      const int bytes = (r < rows_valid) ? kvalid * 8 : 0;
      const double* src = bytes ? rowptr(p) + kcol : safe;
      if (CH == 2) cp_async_chunk16(s_op + dst0 + p * RPP * 32, src, bytes);
      else cp_async_chunk8(s_op + dst0 + p * RPP * 32, src, bytes);
    }
  }
};

// ------------------------------------------------------------------------------------------------- MMA core
struct WarpTile {
  int wr0, wc0;    // first row / col of the warp inside the CTA tile (multiples of 8)
  int mi, nj;      // fragments owned (0..4 each)
  __device__ __forceinline__ WarpTile(int warp, int rows_valid, int cols_valid) {
    const int fm = (rows_valid + 7) >> 3, fn = (cols_valid + 7) >> 3;
    const int hm = (fm + 1) >> 1, hn = (fn + 1) >> 1;
    const int wr = warp >> 1, wc = warp & 1;
    wr0 = wr ? hm * 8 : 0;
    mi = wr ? fm - hm : hm;
    wc0 = wc ? hn * 8 : 0;
    nj = wc ? fn - hn : hn;
  }
};

// One staged K-tile for a warp owning MI x NJ fragments (compile-time, so no predicated DMMA and no WARPSYNC):
// nk4 k-steps of MI*NJ DMMA.8x8x4; the fragments of step ks+1 are fetched while step ks issues.
template <int MI, int NJ>
__device__ __forceinline__ void mma_step(const double (&a)[MI], const double (&b)[NJ], double (&acc)[4][4][2]) {
#pragma unroll
  for (int i = 0; i < MI; ++i)
#pragma unroll
    for (int j = 0; j < NJ; ++j) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
}
template <int MI, int NJ>
__device__ __forceinline__ void load_frags(const double* px, const double* py, int ks, double (&a)[MI], double (&b)[NJ]) {
#pragma unroll
  for (int i = 0; i < MI; ++i) a[i] = px[ks * TILE * 4 + i * 32];
#pragma unroll
  for (int j = 0; j < NJ; ++j) b[j] = py[ks * TILE * 4 + j * 32];
}
template <int MI, int NJ>
__device__ __forceinline__ void mma_stage(const double* px, const double* py, double (&acc)[4][4][2], int nk4) {
  double a0[MI], b0[NJ], a1[MI], b1[NJ];
  load_frags<MI, NJ>(px, py, 0, a0, b0);
  if (nk4 == 4) {                       // the common case: straight-line, no predication, no WARPSYNC
    load_frags<MI, NJ>(px, py, 1, a1, b1);
    mma_step<MI, NJ>(a0, b0, acc);
    load_frags<MI, NJ>(px, py, 2, a0, b0);
    mma_step<MI, NJ>(a1, b1, acc);
    load_frags<MI, NJ>(px, py, 3, a1, b1);
    mma_step<MI, NJ>(a0, b0, acc);
    mma_step<MI, NJ>(a1, b1, acc);
  } else {                              // ragged K tail of a segment (1..3 k-steps)
    mma_step<MI, NJ>(a0, b0, acc);
    for (int ks = 1; ks < nk4; ++ks) {
      load_frags<MI, NJ>(px, py, ks, a0, b0);
      mma_step<MI, NJ>(a0, b0, acc);
    }
  }
}

// Store the warp's accumulators: element (row, col) of the CTA tile goes to dst[row*ld + col]; rowscale(row) multiplies.
template <class RowScale>
__device__ __forceinline__ void store_tile(double* dst, int ld, int rows_valid, int cols_valid,
                                           const double (&acc)[4][4][2], const WarpTile& w, int lane, RowScale rowscale) {
  const int g = lane >> 2, q = lane & 3;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int row = w.wr0 + 8 * i + g;
    if (i >= w.mi || row >= rows_valid) continue;
    const double sc = rowscale(row);
    double* drow = dst + (int64_t)row * ld;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int col = w.wc0 + 8 * j + 2 * q;
      if (j >= w.nj || col >= cols_valid) continue;
      const double v0 = acc[i][j][0] * sc, v1 = acc[i][j][1] * sc;
      double* p = drow + col;
      if (col + 1 < cols_valid) {
        if ((reinterpret_cast<uintptr_t>(p) & 15) == 0) *reinterpret_cast<double2*>(p) = make_double2(v0, v1);
        else { p[0] = v0; p[1] = v1; }
      } else {
        p[0] = v0;
      }
    }
  }
}

// Which tile quadrant consumer warp 0 takes.  Consumer warp w sits on SM sub-partition w, and with odd fragment counts
// the quadrants carry unequal DMMA counts (e.g. 16/12/12/9), so co-resident CTAs must not all put their heavy
// quadrant on the same sub-partition.  CTAs are dealt to SMs round-robin (148 = 0 mod 4), hence a hash, not bid & 3.
__device__ __forceinline__ int quadrant_rotation(unsigned bid) { return (int)((bid * 2654435761u) >> 30); }

// Shared-memory carve-up: NSTAGE stages of [X tile | Y tile], then the barriers and (P1) the row-pointer table.
struct SmemLayout {
  uint32_t base;                                   // shared-window address of stage 0
  __device__ __forceinline__ uint32_t stage(int s) const { return base + s * STAGE_DOUBLES * 8; }
  __device__ __forceinline__ uint32_t full(int s) const { return base + NSTAGE * STAGE_DOUBLES * 8 + s * 8; }
  __device__ __forceinline__ uint32_t empty(int s) const { return base + NSTAGE * STAGE_DOUBLES * 8 + (NSTAGE + s) * 8; }
};
__device__ __forceinline__ void init_barriers(const SmemLayout& sm, int tid) {
  if (tid == 0) {
    for (int s = 0; s < NSTAGE; ++s) { mbar_init(sm.full(s), 32); mbar_init(sm.empty(s), NCONS); }
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();
}


// Consumer main loop for a warp owning MI x NJ fragments.  seq.next() returns the number of k-steps (1..4) of the
// next staged K-tile, or 0 when the unit is done.  Idle warps (MI == 0) only hand the stages back.
template <int MI, int NJ, class Seq>
__device__ __forceinline__ void consume(const double* smem, const SmemLayout& sm, Seq& seq, double (&acc)[4][4][2],
                                        const WarpTile& w, int lane, bool skip_mma) {
  int stage = 0;
  uint32_t phase = 0;
  const int xoff = w.wr0 * 4 + lane, yoff = 4 * TILE * 4 + w.wc0 * 4 + lane;
  for (int nk4 = seq.next(); nk4 > 0; nk4 = seq.next()) {
    mbar_wait(sm.full(stage), phase);
    if (MI > 0 && !skip_mma) {
      const double* st = smem + stage * STAGE_DOUBLES;
      mma_stage<(MI > 0 ? MI : 1), (NJ > 0 ? NJ : 1)>(st + xoff, st + yoff, acc, nk4);
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(sm.empty(stage));
    if (++stage == NSTAGE) { stage = 0; phase ^= 1; }
  }
}

template <class Seq>
__device__ __forceinline__ void consume_dispatch(const double* smem, const SmemLayout& sm, Seq& seq,
                                                 double (&acc)[4][4][2], const WarpTile& w, int lane, bool skip_mma) {
#define HPSI_CASE(MI, NJ) case MI * 5 + NJ: consume<MI, NJ>(smem, sm, seq, acc, w, lane, skip_mma); break;
  switch ((w.nj > 0 ? w.mi : 0) * 5 + (w.mi > 0 ? w.nj : 0)) {
    HPSI_CASE(1, 1) HPSI_CASE(1, 2) HPSI_CASE(1, 3) HPSI_CASE(1, 4)
    HPSI_CASE(2, 1) HPSI_CASE(2, 2) HPSI_CASE(2, 3) HPSI_CASE(2, 4)
    HPSI_CASE(3, 1) HPSI_CASE(3, 2) HPSI_CASE(3, 3) HPSI_CASE(3, 4)
    HPSI_CASE(4, 1) HPSI_CASE(4, 2) HPSI_CASE(4, 3) HPSI_CASE(4, 4)
    default: consume<0, 0>(smem, sm, seq, acc, w, lane, skip_mma); break;
  }
#undef HPSI_CASE
}

// ------------------------------------------------------------------------------------------------ P1 kernel
// One CTA = one P1Unit: C[R0.., j0..] = coef(row) * sum_k X[R,k] Y[j,k], X rows stacked over the group's terms
// (order 1: A_t rows; order 2: B_t rows), Y = padded psi^T (order 1) or padded psi (order 2) block of the source.
template <int CH>
__global__ void __launch_bounds__(NTHREADS, 3) p1_kernel(DevSchedule d) {
  extern __shared__ __align__(16) double smem[];
  const P1Unit u = d.p1[blockIdx.x];
  const Group g = d.groups[u.group];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  SmemLayout sm{(uint32_t)__cvta_generic_to_shared(smem)};
  const double** rowtab = reinterpret_cast<const double**>(smem + NSTAGE * STAGE_DOUBLES + 2 * NSTAGE);
  init_barriers(sm, tid);
  const int ntiles = (g.K1 + KT - 1) / KT;

  if (wid == NCONS) {
    // ---------------- producer warp
    const double* xbase = (g.order == 1) ? d.a : d.b;
    const double* ybase = d.ws + g.y1_off + (int64_t)u.j0 * g.ldy1;
    for (int r = lane; r < TILE; r += 32) {                 // row-pointer table of the stacked X rows
      const double* ptr = ybase;
      if (r < u.rows_valid) {
        const int R = u.R0 + r;
        const int ti = R / g.rows, x = R - ti * g.rows;
        const Seg* sg = d.segs + g.seg0 + ti;
        ptr = xbase + sg->p1_off + (int64_t)x * sg->p1_ld;
      }
      rowtab[r] = ptr;
    }
    __syncwarp();
    const Stager<CH> st(lane);
    const double* yrow0 = ybase + (int64_t)st.r0 * g.ldy1;
    const int64_t ystep = (int64_t)Stager<CH>::RPP * g.ldy1;
    int stage = 0;
    uint32_t phase = 1;
    for (int t = 0; t < ntiles; ++t) {
      mbar_wait(sm.empty(stage), phase);
      const uint32_t sx = sm.stage(stage), sy = sx + 4 * TILE * 4 * 8;
      if (d.debug != 1) {
        st.load(sx, [&](int p) { return rowtab[st.r0 + p * Stager<CH>::RPP]; }, u.rows_valid, ybase, t * KT, g.K1);
        st.load(sy, [&](int p) { return yrow0 + p * ystep; }, u.cols_valid, ybase, t * KT, g.K1);
      }
      cp_async_mbar_arrive(sm.full(stage));
      if (++stage == NSTAGE) { stage = 0; phase ^= 1; }
    }
    cp_async_wait_all();
    return;
  }

  // ------------------ consumer warps
  const int warp = (wid + quadrant_rotation(blockIdx.x)) & 3;
  const WarpTile w(warp, u.rows_valid, u.cols_valid);
  double acc[4][4][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
  struct Seq1 {
    int K, t;
    __device__ __forceinline__ int next() {
      int n = (K - t * KT + 3) >> 2;
      ++t;
      return n > 4 ? 4 : (n < 0 ? 0 : n);
    }
  } seq{g.K1, 0};
  consume_dispatch(smem, sm, seq, acc, w, lane, d.debug == 2);
  double* dst = d.ws + g.ws_off + (int64_t)u.R0 * g.ldw + u.j0;
  store_tile(dst, g.ldw, u.rows_valid, u.cols_valid, acc, w, lane, [&](int row) {
    const int ti = (u.R0 + row) / g.rows;
    return d.segs[g.seg0 + ti].coef;
  });
}

// ------------------------------------------------------------------------------------------------ P2 kernel
// One CTA = one P2Unit: partial[i0.., j0..] = sum over the unit's runs, segs and k of X[i,k] Y[j,k]
// (order 1: X = T_t from the workspace, Y = B_t; order 2: X = A_t, Y = U_t^T from the workspace).
struct KIter {                 // walks (run, seg, kappa) in K-tile steps
  const Run* runs;
  int run, run_end, seg, seg_end, K, kappa, ldw, order;
  bool valid;
  __device__ __forceinline__ void open_run() {
    const Run r = runs[run];
    seg = r.seg_begin; seg_end = r.seg_end; K = r.K; ldw = r.ldw; order = r.order; kappa = 0;
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

template <int CH>
__global__ void __launch_bounds__(NTHREADS, 3) p2_kernel(DevSchedule d) {
  extern __shared__ __align__(16) double smem[];
  const P2Unit u = d.p2[blockIdx.x];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  SmemLayout sm{(uint32_t)__cvta_generic_to_shared(smem)};
  init_barriers(sm, tid);
  KIter it(d.runs, u.run_begin, u.run_end);

  if (wid == NCONS) {
    // ---------------- producer warp
    const Stager<CH> st(lane);
    const double *xrow0 = nullptr, *yrow0 = nullptr, *xsafe = nullptr, *ysafe = nullptr;
    int64_t xstep = 0, ystep = 0;
    auto open_seg = [&]() {
      const Seg* sg = d.segs + it.seg;
      const int64_t p2_off = sg->p2_off, ws_off = sg->ws_off;
      const int p2_ld = sg->p2_ld;
      if (it.order == 1) {
        xsafe = d.ws + ws_off + (int64_t)u.i0 * it.ldw;
        xrow0 = xsafe + (int64_t)st.r0 * it.ldw;
        xstep = (int64_t)Stager<CH>::RPP * it.ldw;
        ysafe = d.b + p2_off + (int64_t)u.j0 * p2_ld;
        yrow0 = ysafe + (int64_t)st.r0 * p2_ld;
        ystep = (int64_t)Stager<CH>::RPP * p2_ld;
      } else {
        xsafe = d.a + p2_off + (int64_t)u.i0 * p2_ld;
        xrow0 = xsafe + (int64_t)st.r0 * p2_ld;
        xstep = (int64_t)Stager<CH>::RPP * p2_ld;
        ysafe = d.ws + ws_off + (int64_t)u.j0 * it.ldw;
        yrow0 = ysafe + (int64_t)st.r0 * it.ldw;
        ystep = (int64_t)Stager<CH>::RPP * it.ldw;
      }
    };
    if (it.valid) open_seg();
    int stage = 0;
    uint32_t phase = 1;
    while (it.valid) {
      mbar_wait(sm.empty(stage), phase);
      const uint32_t sx = sm.stage(stage), sy = sx + 4 * TILE * 4 * 8;
      if (d.debug != 1) {
        st.load(sx, [&](int p) { return xrow0 + p * xstep; }, u.rows_valid, xsafe, it.kappa, it.K);
        st.load(sy, [&](int p) { return yrow0 + p * ystep; }, u.cols_valid, ysafe, it.kappa, it.K);
      }
      cp_async_mbar_arrive(sm.full(stage));
      if (it.advance()) open_seg();
      if (++stage == NSTAGE) { stage = 0; phase ^= 1; }
    }
    cp_async_wait_all();
    return;
  }

  // ------------------ consumer warps
  const int warp = (wid + quadrant_rotation(blockIdx.x)) & 3;
  const WarpTile w(warp, u.rows_valid, u.cols_valid);
  double acc[4][4][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
  struct Seq2 {
    KIter& it;
    __device__ __forceinline__ int next() {
      if (!it.valid) return 0;
      const int n = it.nk4();
      it.advance();
      return n;
    }
  } seq{it};
  consume_dispatch(smem, sm, seq, acc, w, lane, d.debug == 2);
  store_tile(d.ws + u.out_off, u.ldo, u.rows_valid, u.cols_valid, acc, w, lane, [](int) { return 1.0; });
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
  if ((e = cudaFuncSetAttribute(p1_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES))) return e;
  if ((e = cudaFuncSetAttribute(p1_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES))) return e;
  if ((e = cudaFuncSetAttribute(p2_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES))) return e;
  if ((e = cudaFuncSetAttribute(p2_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES))) return e;
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
void launch_p1(const DevSchedule& d, bool aligned16, cudaStream_t st) {
  if (d.n_p1 == 0) return;
  if (aligned16) p1_kernel<2><<<d.n_p1, NTHREADS, SMEM_BYTES, st>>>(d);
  else p1_kernel<1><<<d.n_p1, NTHREADS, SMEM_BYTES, st>>>(d);
}
void launch_p2(const DevSchedule& d, bool aligned16, cudaStream_t st) {
  if (d.n_p2 == 0) return;
  if (aligned16) p2_kernel<2><<<d.n_p2, NTHREADS, SMEM_BYTES, st>>>(d);
  else p2_kernel<1><<<d.n_p2, NTHREADS, SMEM_BYTES, st>>>(d);
}
void launch_reduce(const DevSchedule& d, double* out, cudaStream_t st) {
  if (d.n_blocks > 0) reduce_kernel<<<elem_grid(d), 256, 0, st>>>(d, out);
}
void launch_diag(const DevSchedule& d, double* diag, cudaStream_t st) {
  if (d.n_blocks > 0) diag_kernel<<<elem_grid(d), 256, 0, st>>>(d, diag);
}

}  // namespace hpsi
