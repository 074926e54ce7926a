// Device helpers shared by the GEMM kernels (kernels.cu: blocks stored plainly; kernels_paired.cu: plans with blocks
// stored transposed): PTX wrappers (mbarrier, TMA, cp.async, DMMA), the shared-memory carve-up and the stage ring.
#pragma once
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

// fetch a tensor map into the TMA unit's descriptor cache ahead of its first use (short segments change maps every 2-4 stages)
__device__ __forceinline__ void tma_prefetch_desc(const void* tmap) {
  asm volatile("prefetch.tensormap [%0];\n" ::"l"(tmap) : "memory");
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

// Same accumulators stored transposed: element (row, col) of the CTA tile goes to dst[col*ld + row]  (operator update,
// rotate.cu: the first GEMM leaves T^T, the second A').  The 8 lane groups of a store cover 8 consecutive rows = 64
// contiguous bytes of each of 4 destination rows.
template <int MI, int NJ>
__device__ __forceinline__ void store_tile_t(double* dst, int ld, int rows_valid, int cols_valid,
                                             const double (&acc)[MI][NJ][2], const WarpTile& w, int lane) {
  const int pg = frag_perm(lane >> 2), pc = frag_perm(2 * (lane & 3));
#pragma unroll
  for (int i = 0; i < MI; ++i) {
    const int row = w.wr0 + 8 * i + pg;
    if (row >= rows_valid) continue;
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
      const int col = w.wc0 + 8 * j + pc;
      if (col < cols_valid) dst[(int64_t)col * ld + row] = acc[i][j][0];
      if (col + 2 < cols_valid) dst[(int64_t)(col + 2) * ld + row] = acc[i][j][1];
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

}  // namespace hpsi
