// sm_100a kernels of hpsi_apply: prep (padded psi, psi^T), P1 (stacked first GEMM), P2 (segmented-K second GEMM
// with split-K partials), reduce (ordered sum of partials), diag.  See kernels.cuh / plan.h for the vocabulary.
#include "kernels.cuh"

namespace hpsi {

// ----------------------------------------------------------------------------------------------- PTX helpers
__device__ __forceinline__ void cp_async_chunk16(uint32_t dst, const void* src, int bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(dst), "l"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cp_async_chunk8(uint32_t dst, const void* src, int bytes) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(dst), "l"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

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
template <int CH>
struct Stager {
  static constexpr int CPR = KT / CH;            // chunks per row
  static constexpr int RPP = NTHREADS / CPR;     // rows per pass
  static constexpr int PASSES = TILE / RPP;
  int r0, kc;
  uint32_t dst0;                                 // byte offset inside an operand's stage
  __device__ __forceinline__ Stager(int tid) {
    const int c = tid % CPR;
    r0 = tid / CPR;
    kc = c * CH;
    dst0 = (uint32_t)((((kc >> 2) * TILE + r0) * 4 + (kc & 3)) * 8);
  }
  // rows r0 + p*RPP of the operand; rowptr(p) = pointer to (row, k=0) of that row in global memory
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

__device__ __forceinline__ void mma_stage(const double* sx, const double* sy, double (&acc)[4][4][2], int nk4,
                                          const WarpTile& w, int lane) {
  const double* px = sx + w.wr0 * 4 + lane;
  const double* py = sy + w.wc0 * 4 + lane;
  if (w.mi == 4 && w.nj == 4) {
#pragma unroll 1
    for (int ks = 0; ks < nk4; ++ks) {
      double a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) { a[i] = px[ks * TILE * 4 + i * 32]; b[i] = py[ks * TILE * 4 + i * 32]; }
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
    }
  } else {
#pragma unroll 1
    for (int ks = 0; ks < nk4; ++ks) {
      double a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) { a[i] = px[ks * TILE * 4 + i * 32]; b[i] = py[ks * TILE * 4 + i * 32]; }
#pragma unroll
      for (int i = 0; i < 4; ++i)
        if (i < w.mi) {
#pragma unroll
          for (int j = 0; j < 4; ++j)
            if (j < w.nj) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
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

// ------------------------------------------------------------------------------------------------ P1 kernel
// One CTA = one P1Unit: C[R0.., j0..] = coef(row) * sum_k X[R,k] Y[j,k], X rows stacked over the group's terms
// (order 1: A_t rows; order 2: B_t rows), Y = padded psi^T (order 1) or padded psi (order 2) block of the source.
template <int CH>
__global__ void __launch_bounds__(NTHREADS, 4) p1_kernel(DevSchedule d) {
  extern __shared__ __align__(16) double smem[];
  const P1Unit u = d.p1[blockIdx.x];
  const Group g = d.groups[u.group];
  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = ((tid >> 5) + blockIdx.x) & 3;          // rotate so light edge warps spread over the 4 SMSPs
  const double* xbase = (g.order == 1) ? d.a : d.b;
  const double* ybase = d.ws + g.y1_off + (int64_t)u.j0 * g.ldy1;

  const Stager<CH> st(tid);
  const double* xrow[Stager<CH>::PASSES];
#pragma unroll
  for (int p = 0; p < Stager<CH>::PASSES; ++p) {
    const int r = st.r0 + p * Stager<CH>::RPP;
    xrow[p] = ybase;
    if (r < u.rows_valid) {
      const int R = u.R0 + r;
      const int ti = R / g.rows, x = R - ti * g.rows;
      const Seg* sg = d.segs + g.seg0 + ti;
      xrow[p] = xbase + sg->p1_off + (int64_t)x * sg->p1_ld;
    }
  }
  const double* yrow0 = ybase + (int64_t)st.r0 * g.ldy1;
  const int64_t ystep = (int64_t)Stager<CH>::RPP * g.ldy1;
  const uint32_t s0 = (uint32_t)__cvta_generic_to_shared(smem);

  auto load = [&](int stage, int kappa) {
    const uint32_t sx = s0 + stage * STAGE_DOUBLES * 8, sy = sx + 4 * TILE * 4 * 8;
    st.load(sx, [&](int p) { return xrow[p]; }, u.rows_valid, ybase, kappa, g.K1);
    st.load(sy, [&](int p) { return yrow0 + p * ystep; }, u.cols_valid, ybase, kappa, g.K1);
  };

  const WarpTile w(warp, u.rows_valid, u.cols_valid);
  double acc[4][4][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

  const int ntiles = (g.K1 + KT - 1) / KT;
#pragma unroll
  for (int s = 0; s < NSTAGE - 1; ++s) {
    if (s < ntiles) load(s, s * KT);
    cp_async_commit();
  }
  for (int t = 0; t < ntiles; ++t) {
    cp_async_wait<NSTAGE - 2>();
    __syncthreads();
    const int nt = t + NSTAGE - 1;
    if (nt < ntiles) load(nt % NSTAGE, nt * KT);
    cp_async_commit();
    const double* sx = smem + (t % NSTAGE) * STAGE_DOUBLES;
    int nk4 = (g.K1 - t * KT + 3) >> 2;
    nk4 = nk4 > 4 ? 4 : nk4;
    mma_stage(sx, sx + 4 * TILE * 4, acc, nk4, w, lane);
  }
  cp_async_wait<0>();

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
__global__ void __launch_bounds__(NTHREADS, 4) p2_kernel(DevSchedule d) {
  extern __shared__ __align__(16) double smem[];
  const P2Unit u = d.p2[blockIdx.x];
  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = ((tid >> 5) + blockIdx.x) & 3;
  const Stager<CH> st(tid);
  const uint32_t s0 = (uint32_t)__cvta_generic_to_shared(smem);

  KIter prod(d.runs, u.run_begin, u.run_end), cons(d.runs, u.run_begin, u.run_end);
  const double *xrow0 = nullptr, *yrow0 = nullptr, *xsafe = nullptr, *ysafe = nullptr;
  int64_t xstep = 0, ystep = 0;
  auto open_seg = [&]() {
    const Seg* sg = d.segs + prod.seg;
    const int64_t p2_off = sg->p2_off, ws_off = sg->ws_off;
    const int p2_ld = sg->p2_ld;
    if (prod.order == 1) {
      xsafe = d.ws + ws_off + (int64_t)u.i0 * prod.ldw;
      xrow0 = xsafe + (int64_t)st.r0 * prod.ldw;
      xstep = (int64_t)Stager<CH>::RPP * prod.ldw;
      ysafe = d.b + p2_off + (int64_t)u.j0 * p2_ld;
      yrow0 = ysafe + (int64_t)st.r0 * p2_ld;
      ystep = (int64_t)Stager<CH>::RPP * p2_ld;
    } else {
      xsafe = d.a + p2_off + (int64_t)u.i0 * p2_ld;
      xrow0 = xsafe + (int64_t)st.r0 * p2_ld;
      xstep = (int64_t)Stager<CH>::RPP * p2_ld;
      ysafe = d.ws + ws_off + (int64_t)u.j0 * prod.ldw;
      yrow0 = ysafe + (int64_t)st.r0 * prod.ldw;
      ystep = (int64_t)Stager<CH>::RPP * prod.ldw;
    }
  };
  auto load = [&](int stage) {
    const uint32_t sx = s0 + stage * STAGE_DOUBLES * 8, sy = sx + 4 * TILE * 4 * 8;
    st.load(sx, [&](int p) { return xrow0 + p * xstep; }, u.rows_valid, xsafe, prod.kappa, prod.K);
    st.load(sy, [&](int p) { return yrow0 + p * ystep; }, u.cols_valid, ysafe, prod.kappa, prod.K);
  };

  const WarpTile w(warp, u.rows_valid, u.cols_valid);
  double acc[4][4][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

  if (prod.valid) open_seg();
#pragma unroll
  for (int s = 0; s < NSTAGE - 1; ++s) {
    if (prod.valid) {
      load(s);
      if (prod.advance()) open_seg();
    }
    cp_async_commit();
  }
  int stage = 0, pstage = NSTAGE - 1;
  while (cons.valid) {
    cp_async_wait<NSTAGE - 2>();
    __syncthreads();
    if (prod.valid) {
      load(pstage);
      if (prod.advance()) open_seg();
    }
    cp_async_commit();
    const double* sx = smem + stage * STAGE_DOUBLES;
    mma_stage(sx, sx + 4 * TILE * 4, acc, cons.nk4(), w, lane);
    cons.advance();
    stage = (stage + 1 == NSTAGE) ? 0 : stage + 1;
    pstage = (pstage + 1 == NSTAGE) ? 0 : pstage + 1;
  }
  cp_async_wait<0>();

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
