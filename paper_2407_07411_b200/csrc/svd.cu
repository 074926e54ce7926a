// hpsi_truncate (include/hpsi.h "Site update"): the matrix factorisation of a
// DMRG tensor update - SVD of every psi block, global selection of the chi_max largest singular values, left isometries.
//
// One-sided Jacobi (Hestenes) on the ROWS of each block: row i of the working matrix is [ psi_l[i, :] | R[i, :] ] with
// R = 1 at the start; plane rotations make the psi parts mutually orthogonal, the same rotations applied to R
// accumulate J with  J psi_l = S V^T,  i.e. psi_l = J^T S V^T: row i of R is the i-th left singular vector and the norm
// of the psi part its singular value.  Rows are contiguous (the psi layout is row-major), so a rotation streams two
// rows with unit stride.  A block with more rows than columns has linearly dependent rows (the surplus rows would only
// decay linearly, sweep after sweep: measured 22 sweeps instead of 12 on the cyp blocks), so there the vectors are the COLUMNS: the working
// matrix is psi_l^T alone, its converged rows are sigma_j u_j^T and the isometry rows are those rows divided by sigma_j.
//
// Parallel order (block Jacobi by tournament): the rows of a block are cut into chunks of 16 rows; in one kernel launch
// ("round") every CTA owns one PAIR of chunks of one block, chosen by the round-robin (circle) schedule so that all CTAs
// of a round touch disjoint rows.  A visit does not rotate the 32 rows themselves pair by pair (that streams two rows
// through shared memory three times per pair - the first version of this kernel was bound by shared-memory bandwidth):
// it forms their 32 x 32 Gram matrix G on the tensor pipe, runs the visit's plane rotations on G (both sides) while
// accumulating their product Q, and applies Q to the rows once, again on the tensor pipe (svd_round_kernel).  The pairs,
// their order, the rotation formula and the threshold are those of the row-by-row method: the first round of a block's
// sweep does all pairs inside the two chunks, the others only the cross pairs, so a sweep visits every row pair of the
// block exactly once.  Sweeps repeat until one makes no rotation (device counter of rotations; the only atomic, not on
// data).  Every psi block is processed in the same launches.  FP64 throughout; the result is bitwise reproducible.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <mutex>
#include <numeric>
#include <vector>

#include "plan_dev.h"

namespace hpsi {

struct SvdBlk {
  int64_t w_off;        // working matrix nv x L in the SVD workspace
  int64_t psi_off;      // block in psi (dense rows x cols)
  int32_t rows, cols;   // of the block whose ROW space is truncated: the psi block (left side) or its transpose (right side)
  int32_t nv, vlen;     // vectors orthogonalised and their length: (rows, cols) if rows <= cols, else (cols, rows)
  int32_t tall;         // 1: rows > cols, the working matrix is the transposed block without the R part
  int32_t pcols, rt;    // leading dimension of the block in psi; rt = 1: working vector i, element j is psi[j][i]
  int32_t L;            // leading dimension: vlen (+ rows for the R part) rounded up to 4
  int32_t nce;          // chunks, padded to an even count >= 2
  int32_t cta0;         // first CTA of this block in a round
  int32_t row0;         // first row in the concatenated singular-value array
  double floor2;        // rows with squared norm <= floor2 count as zero (1e-27 x the block's squared Frobenius norm)
};

// working matrix <- [psi block | identity]; floor2 of the block from its Frobenius norm (one CTA per block row range)
__global__ void svd_init_kernel(SvdBlk* blk, const double* __restrict__ psi, double* __restrict__ w) {
  pdl_wait();
  const SvdBlk B = blk[blockIdx.y];
  for (int i = blockIdx.x; i < B.nv; i += gridDim.x) {
    double* row = w + B.w_off + (int64_t)i * B.L;
    for (int j = threadIdx.x; j < B.L; j += blockDim.x) {
      double v = 0.0;
      if (j < B.vlen) v = B.rt ? psi[B.psi_off + (int64_t)j * B.pcols + i] : psi[B.psi_off + (int64_t)i * B.pcols + j];
      else if (!B.tall && j - B.vlen == i) v = 1.0;
      row[j] = v;
    }
  }
}
// squared Frobenius norm of each block in a fixed order (one CTA per block, tree reduction)
__global__ void svd_norm_kernel(SvdBlk* blk, const double* __restrict__ psi) {
  pdl_wait();
  __shared__ double red[256];
  SvdBlk& B = blk[blockIdx.x];
  const int64_t n = (int64_t)B.rows * B.cols;
  double s = 0.0;
  for (int64_t e = threadIdx.x; e < n; e += blockDim.x) { const double v = psi[B.psi_off + e]; s += v * v; }
  red[threadIdx.x] = s;
  __syncthreads();
  for (int k = 128; k > 0; k >>= 1) {
    if ((int)threadIdx.x < k) red[threadIdx.x] += red[threadIdx.x + k];
    __syncthreads();
  }
  if (threadIdx.x == 0) B.floor2 = 1e-27 * red[0];
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

constexpr int SV_B = 16;             // rows per chunk
constexpr int SV_M = 2 * SV_B;       // rows one CTA orthogonalises per visit (a chunk pair)
constexpr int SV_KC = 32;            // columns of the psi part staged per Gram step (512 threads x 2 doubles)
constexpr int SV_THREADS = 512;      // 16 warps: one Gram fragment, one row pair of a rotation step, one (row half, column block) each

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

struct SvdSmem {
  double G[SV_M][SV_M + 1];          // Gram matrix of the psi parts of the 32 rows, rotated two-sidedly
  double Q[SV_M][SV_M + 1];          // product of the visit's rotations: the rows become Q X
  double stage[2][SV_M][SV_KC + 4];  // psi part, one K-chunk of all 32 rows (double buffered)
  double cs[SV_B][2];                // rotations of the current step
};

// One round: CTA = (block, chunk pair of the round-robin schedule).  Block Jacobi on the tensor pipe:
//   1. G = X_psi X_psi^T for the 32 rows of the chunk pair (DMMA, the rows streamed once through shared memory);
//   2. one cyclic pass of plane rotations over the row pairs of the visit, applied to G from both sides (32-long vectors
//      in shared memory instead of the rows themselves) and accumulated in Q - same pairs, same order, same rotation
//      formula and threshold as rotating the rows one pair at a time.  One warp per pair: the chain square root ->
//      division -> reciprocal square root of a rotation is ~600 clk, and 16 (cross pairs) or 31 (all pairs) such steps
//      in sequence are the critical path of a visit;
//   3. X <- Q X over all L columns (DMMA, every element read and written once).
// Shared-memory traffic per visit drops from ~93 passes over the 32 rows (31 inner rounds x 3) to 2 passes through
// global memory / L2.
__global__ void __launch_bounds__(SV_THREADS, 2) svd_round_kernel(const SvdBlk* __restrict__ blk, const int32_t* __restrict__ cta_blk,
                                                               int round, double* __restrict__ w, int* __restrict__ flag) {
  pdl_wait();
  __shared__ SvdSmem sm;
  const SvdBlk B = blk[cta_blk[blockIdx.x]];
  const int k = blockIdx.x - B.cta0;
  const int n1 = B.nce - 1;
  const int rr = round % n1;
  int ci, cj;                                            // the two chunks of this CTA (circle method)
  if (k == 0) { ci = n1; cj = rr; }
  else { ci = (rr + k) % n1; cj = (rr - k + n1) % n1; }
  if (ci > cj) { const int t = ci; ci = cj; cj = t; }
  const bool full = (rr == 0);                           // first round of the block's sweep: pairs inside the chunks too
  const int ni = max(0, min(SV_B, B.nv - ci * SV_B)), nj = max(0, min(SV_B, B.nv - cj * SV_B));
  if (ni + nj < 2 || (!full && (ni == 0 || nj == 0))) return;
  const int L = B.L, tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int g = lane >> 2, q = lane & 3;
  // slot s < 16 holds row ci*16 + s, slot 16 + s holds row cj*16 + s
  auto valid = [&](int slot) { return slot < SV_B ? slot < ni : slot - SV_B < nj; };
  auto grow = [&](int slot) -> double* {
    const int row = slot < SV_B ? ci * SV_B + slot : cj * SV_B + (slot - SV_B);
    return w + B.w_off + (int64_t)row * L;
  };

  // ---- 1. Gram matrix: warp wid owns fragment (i, j) = (wid / 4, wid % 4) of the 4 x 4 grid of 8 x 8 fragments
  {
    const int fi = wid >> 2, fj = wid & 3;
    double acc0 = 0.0, acc1 = 0.0;
    const int lrow = tid >> 4, lc = (tid & 15) * 2;      // this thread stages 2 consecutive columns of one row
    const bool lvalid = valid(lrow);
    const double* lsrc = grow(lrow);
    double v0, v1;
    auto fetch = [&](int kc) {
      const int c = kc + lc;
      v0 = (lvalid && c < B.vlen) ? lsrc[c] : 0.0;
      v1 = (lvalid && c + 1 < B.vlen) ? lsrc[c + 1] : 0.0;
    };
    const int nchunk = (B.vlen + SV_KC - 1) / SV_KC;
    fetch(0);
    for (int ch = 0; ch < nchunk; ++ch) {
      double (*st)[SV_KC + 4] = sm.stage[ch & 1];
      st[lrow][lc] = v0;
      st[lrow][lc + 1] = v1;
      __syncthreads();                                   // chunk ch staged; everybody is past the DMMAs of chunk ch - 2
      if (ch + 1 < nchunk) fetch((ch + 1) * SV_KC);
#pragma unroll
      for (int ks = 0; ks < SV_KC / 4; ++ks)
        dmma884(acc0, acc1, st[8 * fi + g][4 * ks + q], st[8 * fj + g][4 * ks + q]);
    }
    sm.G[8 * fi + g][8 * fj + 2 * q] = acc0;
    sm.G[8 * fi + g][8 * fj + 2 * q + 1] = acc1;
    for (int e = tid; e < SV_M * SV_M; e += SV_THREADS) sm.Q[e >> 5][e & 31] = ((e >> 5) == (e & 31)) ? 1.0 : 0.0;
  }
  __syncthreads();

  // ---- 2. one pass over the row pairs of the visit, on G (two-sided) and Q: warp wid = pair wid of the step
  // rotate when |<x_p,x_q>| > tol |x_p||x_q| with tol = cols * 2^-53, the threshold LAPACK's Jacobi SVD (dgesvj) uses:
  // a dot product of `cols` terms cannot resolve angles below ~sqrt(cols) * 2^-53, and a tighter test only makes
  // rounding noise trigger further sweeps
  const double tol = 1.1102230246251565e-16 * (double)max(B.vlen, 8);
  int rotated = 0;
  const int np = SV_M - 1;
  const int inner = full ? np : SV_B;
  for (int s = 0; s < inner; ++s) {
    int p, qq;
    if (full) {
      if (wid == 0) { p = np; qq = s; }
      else { p = (s + wid) % np; qq = (s - wid + np) % np; }
    } else {
      p = wid; qq = SV_B + (wid + s) % SV_B;
    }
    double cs = 1.0, sn = 0.0;
    if (valid(p) && valid(qq)) {
      const double a = sm.G[p][p], b = sm.G[qq][qq], gg = sm.G[p][qq];
      if (a > B.floor2 && b > B.floor2 && gg * gg > tol * tol * a * b) {
        // tan of the smaller rotation angle: t = sign(zeta) / (|zeta| + sqrt(1 + zeta^2)) with zeta = (b - a) / 2g
        const double d = b - a;
        const double t = 2.0 * gg / (d + copysign(sqrt(d * d + 4.0 * gg * gg), d));
        cs = rsqrt(1.0 + t * t);
        sn = cs * t;
        ++rotated;
      }
    }
    __syncwarp();
    if (lane == 0) { sm.cs[wid][0] = cs; sm.cs[wid][1] = sn; }
    if (sn != 0.0) {                                     // rows p, q of G and of Q (this pair's alone)
      const double gp = sm.G[p][lane], gq = sm.G[qq][lane];
      sm.G[p][lane] = cs * gp - sn * gq;
      sm.G[qq][lane] = sn * gp + cs * gq;
      const double qp = sm.Q[p][lane], qv = sm.Q[qq][lane];
      sm.Q[p][lane] = cs * qp - sn * qv;
      sm.Q[qq][lane] = sn * qp + cs * qv;
    }
    __syncthreads();
    if (sn != 0.0) {                                     // columns p, q of G (same warp: its cs / sn are still in registers)
      const double gp = sm.G[lane][p], gq = sm.G[lane][qq];
      sm.G[lane][p] = cs * gp - sn * gq;
      sm.G[lane][qq] = sn * gp + cs * gq;
    }
    __syncthreads();
  }
  const int any = __syncthreads_or(rotated);
  if (!any) return;                                      // nothing rotated: the rows stay as they are

  // ---- 3. X <- Q X over all L columns: warp wid owns row blocks 2h, 2h+1 (h = wid / 8) of the 8-column blocks
  // wid % 8, wid % 8 + 8, ...
  const int h = wid >> 3, wc = wid & 7;
  double qa[2][SV_M / 4];                                // A fragments of Q: row block 2h + i, k-step ks
#pragma unroll
  for (int i = 0; i < 2; ++i)
#pragma unroll
    for (int ks = 0; ks < SV_M / 4; ++ks) qa[i][ks] = sm.Q[8 * (2 * h + i) + g][4 * ks + q];
  const double* brow[SV_M / 4];                          // row 4 ks + q of the visit (B fragment: k = q, n = g)
  bool bval[SV_M / 4];
#pragma unroll
  for (int ks = 0; ks < SV_M / 4; ++ks) { bval[ks] = valid(4 * ks + q); brow[ks] = grow(4 * ks + q); }
  // The two warps that share a column block (wid and wid ^ 8) read all 32 rows of it and write 16 each, so both must have
  // read before either writes: a named barrier of those 64 threads between the loads and the stores.
  const int nblk = (L + 7) / 8, nround = (nblk + 7) / 8;
  for (int rd = 0; rd < nround; ++rd) {
    const int col0 = 8 * (wc + 8 * rd);
    double bf[SV_M / 4];
    const bool cok = col0 + g < L;
#pragma unroll
    for (int ks = 0; ks < SV_M / 4; ++ks) bf[ks] = (bval[ks] && cok) ? brow[ks][col0 + g] : 0.0;
    double acc[2][2] = {{0.0, 0.0}, {0.0, 0.0}};
#pragma unroll
    for (int ks = 0; ks < SV_M / 4; ++ks)
#pragma unroll
      for (int i = 0; i < 2; ++i) dmma884(acc[i][0], acc[i][1], qa[i][ks], bf[ks]);
    asm volatile("bar.sync %0, 64;\n" ::"r"(1 + wc) : "memory");   // the two warps of this column block have both read it
    const int c = col0 + 2 * q;
    if (c < L) {                                         // L is even: the pair (c, c + 1) is inside the row or outside it
#pragma unroll
      for (int i = 0; i < 2; ++i) {
        const int slot = 8 * (2 * h + i) + g;
        if (valid(slot)) *reinterpret_cast<double2*>(grow(slot) + c) = make_double2(acc[i][0], acc[i][1]);
      }
    }
  }
  if (lane == 0 && rotated) atomicAdd(flag, rotated);    // rotations of the sweep (control only, not data)
}

// singular value of every row = norm of its psi part (one warp per row)
__global__ void svd_sigma_kernel(const SvdBlk* __restrict__ blk, const double* __restrict__ w, double* __restrict__ sigma) {
  pdl_wait();
  const SvdBlk B = blk[blockIdx.y];
  const int lane = threadIdx.x & 31, wpb = blockDim.x >> 5;
  for (int i = blockIdx.x * wpb + (threadIdx.x >> 5); i < B.nv; i += gridDim.x * wpb) {
    const double* row = w + B.w_off + (int64_t)i * B.L;
    double a = 0.0;
    for (int j = lane; j < B.vlen; j += 32) a = fma(row[j], row[j], a);
    a = warp_sum(a);
    if (lane == 0) sigma[B.row0 + i] = sqrt(a);
  }
}

struct IsoRow { int64_t src, dst; double scale; int32_t len, pad; };   // kept vector (R part, or row / sigma) -> one row of O_l^T
__global__ void svd_gather_kernel(const IsoRow* __restrict__ rows, int n, const double* __restrict__ w, double* __restrict__ ot) {
  pdl_wait();
  for (int i = blockIdx.x; i < n; i += gridDim.x) {
    const IsoRow r = rows[i];
    for (int j = threadIdx.x; j < r.len; j += blockDim.x) ot[r.dst + j] = w[r.src + j] * r.scale;
  }
}

}  // namespace hpsi

using namespace hpsi;

// Scratch of hpsi_truncate_static: one array per GPU that loads the library, held until the process exits.  In host code
// the name is a host-side stand-in, not a device address: truncate_static_scratch() asks the runtime for the address once
// per device and the kernels get that pointer.
static __device__ __align__(256) unsigned char g_truncate_scratch[HPSI_TRUNCATE_STATIC_BYTES];

static int truncate_static_scratch(char** out) {
  constexpr int MAX_DEVICES = 64;
  static std::mutex mu;
  static char* ptr_of_device[MAX_DEVICES] = {};
  int dev = -1;
  HPSI_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= MAX_DEVICES) { set_error("hpsi_truncate_static: device ordinal out of range"); return HPSI_EINVAL; }
  std::lock_guard<std::mutex> lock(mu);
  if (!ptr_of_device[dev]) {
    void* q = nullptr;
    HPSI_CUDA(cudaGetSymbolAddress(&q, g_truncate_scratch));       // the current device's copy of the array
    if (!q) { set_error("hpsi_truncate_static: cudaGetSymbolAddress returned a null address"); return HPSI_ECUDA; }
    ptr_of_device[dev] = static_cast<char*>(q);
  }
  *out = ptr_of_device[dev];
  return HPSI_OK;
}

// hpsi_truncate / hpsi_truncate_static: the same steps; `static_base` != nullptr takes the device buffers from that array
// (capacity static_bytes) instead of the plan's lazily grown cudaMalloc block.
static int truncate_impl(hpsi_plan_t* p, const double* psi_dev, int32_t side, int32_t chi_max, double eps_discard,
                         double* ot_dev, int32_t* chi_host, double* sigma_host, double* discarded_host, void* cuda_stream,
                         char* static_base, size_t static_bytes) {
  if (!p) { set_error("null plan"); return HPSI_EINVAL; }
  if (p->host_only) { set_error("host-only plan: hpsi_truncate needs a CUDA device (no CPU fallback)"); return HPSI_ESTATE; }
  if (chi_max < 0) { set_error("negative chi_max"); return HPSI_EINVAL; }
  if (side != HPSI_SIDE_LEFT && side != HPSI_SIDE_RIGHT) { set_error("side must be HPSI_SIDE_LEFT or HPSI_SIDE_RIGHT"); return HPSI_EINVAL; }
  if (!chi_host) { set_error("null chi_host"); return HPSI_EINVAL; }
  const Schedule& sc = p->sc;
  const int n_sec = side == HPSI_SIDE_LEFT ? p->n_left : p->n_right;
  for (int i = 0; i < n_sec; ++i) chi_host[i] = 0;
  if (discarded_host) *discarded_host = 0.0;
  const int nB = (int)sc.blocks.size();
  if (nB == 0) return HPSI_OK;
  if (!psi_dev || !ot_dev) { set_error("null psi / ot"); return HPSI_EINVAL; }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);

  // ---- tables (rebuilt per call: a few KB of host work)
  std::vector<SvdBlk> tab(nB);
  int Lmax = 0;
  int64_t wlen = 0;
  int row0 = 0;
  for (int b = 0; b < nB; ++b) {
    const PsiBlk& B = sc.blocks[b];
    SvdBlk& s = tab[b];
    s.w_off = wlen; s.psi_off = B.off; s.pcols = B.cols;
    s.rows = side == HPSI_SIDE_LEFT ? B.rows : B.cols;       // the right side truncates the row space of psi_l^T
    s.cols = side == HPSI_SIDE_LEFT ? B.cols : B.rows;
    s.tall = s.rows > s.cols ? 1 : 0;
    s.rt = s.tall ^ (side == HPSI_SIDE_LEFT ? 0 : 1);
    s.nv = std::min(B.rows, B.cols); s.vlen = std::max(B.rows, B.cols);
    s.L = s.tall ? sector_up(s.vlen) : sector_up(B.rows + B.cols);
    s.row0 = row0; s.floor2 = 0.0;
    row0 += s.nv;
    wlen = (wlen + (int64_t)s.nv * s.L + 15) & ~(int64_t)15;
    Lmax = std::max(Lmax, s.L);
  }
  const int n_rows = row0;
  const int bsz = SV_B;
  int n_cta = 0, rounds = 1;
  std::vector<int32_t> cta_blk;
  for (int b = 0; b < nB; ++b) {
    SvdBlk& s = tab[b];
    int nc = (s.nv + bsz - 1) / bsz;
    nc += nc & 1;
    s.nce = std::max(nc, 2);
    s.cta0 = n_cta;
    n_cta += s.nce / 2;
    for (int k = 0; k < s.nce / 2; ++k) cta_blk.push_back(b);
    rounds = std::max(rounds, s.nce - 1);
  }
  // ---- device buffers (kept on the plan; regrown if a call needs more, e.g. the other side)
  const size_t bytes = (size_t)wlen * 8 + (size_t)n_rows * 8 + tab.size() * sizeof(SvdBlk) + cta_blk.size() * 4 + (size_t)n_rows * sizeof(IsoRow) + 4096;
  if (static_base) {
    if (bytes > static_bytes) {
      char buf[200];
      snprintf(buf, sizeof buf, "hpsi_truncate_static: this plan needs %zu bytes of scratch, the static array holds %zu "
               "(HPSI_TRUNCATE_STATIC_BYTES); use hpsi_truncate", bytes, static_bytes);
      set_error(buf);
      return HPSI_EINVAL;
    }
  } else {
    if (bytes > p->svd_bytes) {
      HPSI_CUDA(cudaStreamSynchronize(st));
      cudaFree(p->d_svd);
      p->d_svd = nullptr;
      p->svd_bytes = 0;
      cudaError_t e = cudaMalloc(&p->d_svd, bytes);
      if (e != cudaSuccess) { cudaGetLastError(); set_error("hpsi_truncate: device workspace allocation failed"); return HPSI_ENOMEM; }
      p->svd_bytes = bytes;
    }
  }
  char* base = static_base ? static_base : static_cast<char*>(p->d_svd);
  size_t cur = 0;
  auto carve = [&](size_t bytes) { char* q = base + cur; cur = (cur + bytes + 255) & ~(size_t)255; return q; };
  double* d_w = reinterpret_cast<double*>(carve((size_t)wlen * 8));
  double* d_sigma = reinterpret_cast<double*>(carve((size_t)n_rows * 8));
  SvdBlk* d_tab = reinterpret_cast<SvdBlk*>(carve(tab.size() * sizeof(SvdBlk)));
  int32_t* d_cta = reinterpret_cast<int32_t*>(carve(cta_blk.size() * 4));
  IsoRow* d_rows = reinterpret_cast<IsoRow*>(carve((size_t)n_rows * sizeof(IsoRow)));
  int* d_flag = reinterpret_cast<int*>(carve(256));
  HPSI_CUDA(cudaMemcpyAsync(d_tab, tab.data(), tab.size() * sizeof(SvdBlk), cudaMemcpyHostToDevice, st));
  HPSI_CUDA(cudaMemcpyAsync(d_cta, cta_blk.data(), cta_blk.size() * 4, cudaMemcpyHostToDevice, st));

  launch_dependent(svd_norm_kernel, dim3(nB), dim3(256), 0, st, d_tab, psi_dev);
  launch_dependent(svd_init_kernel, dim3(dim3(64, nB)), dim3(128), 0, st, d_tab, psi_dev, d_w);
  constexpr int MAX_SWEEPS = 60;
  int sweeps = 0, flag = 1;
  for (; sweeps < MAX_SWEEPS && flag; ++sweeps) {
    HPSI_CUDA(cudaMemsetAsync(d_flag, 0, sizeof(int), st));
    for (int r = 0; r < rounds; ++r)
      launch_dependent(svd_round_kernel, dim3(n_cta), dim3(SV_THREADS), 0, st, d_tab, d_cta, sweeps * rounds + r, d_w, d_flag);
    HPSI_CUDA(cudaMemcpyAsync(&flag, d_flag, sizeof(int), cudaMemcpyDeviceToHost, st));
    HPSI_CUDA(cudaStreamSynchronize(st));
  }
  if (flag) { set_error("hpsi_truncate: Jacobi SVD did not converge"); return HPSI_ESTATE; }
  p->svd_sweeps = sweeps;
  p->svd_launches = sweeps * rounds + 4;
  launch_dependent(svd_sigma_kernel, dim3(dim3(16, nB)), dim3(256), 0, st, d_tab, d_w, d_sigma);
  std::vector<double> sig(n_rows);
  HPSI_CUDA(cudaMemcpyAsync(sig.data(), d_sigma, (size_t)n_rows * 8, cudaMemcpyDeviceToHost, st));
  HPSI_CUDA(cudaStreamSynchronize(st));

  // ---- host: order every block's rows by descending singular value, global selection (reading R3)
  struct Cand { double s; int blk, rank, row; };
  std::vector<Cand> cand;
  cand.reserve(n_rows);
  double smax = 0.0;
  int64_t out_row0 = 0;                                // sigma_host holds d_left entries per block
  for (int b = 0; b < nB; ++b) {
    const SvdBlk& s = tab[b];
    std::vector<int> ord(s.nv);
    std::iota(ord.begin(), ord.end(), 0);
    std::stable_sort(ord.begin(), ord.end(), [&](int x, int y) { return sig[s.row0 + x] > sig[s.row0 + y]; });
    for (int k = 0; k < s.rows; ++k) {
      const double v = k < s.nv ? sig[s.row0 + ord[k]] : 0.0;
      if (sigma_host) sigma_host[out_row0 + k] = v;
      if (k < s.nv) { cand.push_back({v, b, k, ord[k]}); smax = std::max(smax, v); }
    }
    out_row0 += s.rows;
  }
  std::stable_sort(cand.begin(), cand.end(), [](const Cand& x, const Cand& y) {
    if (x.s != y.s) return x.s > y.s;
    if (x.blk != y.blk) return x.blk < y.blk;
    return x.rank < y.rank;
  });
  std::vector<std::vector<int>> kept(nB);
  std::vector<char> is_kept(cand.size(), 0);
  int limit = chi_max;
  if (eps_discard >= 0.0) {                            // reading R6: smallest count whose discarded weight is <= eps_discard
    double tail = 0.0;                                 // weight discarded when the first i are kept, summed smallest first
    size_t i = cand.size();
    while (i > 0 && tail + cand[i - 1].s * cand[i - 1].s <= eps_discard) { tail += cand[i - 1].s * cand[i - 1].s; --i; }
    limit = std::min<int64_t>(chi_max, (int64_t)i);
  }
  int nk = 0;
  for (size_t i = 0; i < cand.size(); ++i) {
    if (nk >= limit || cand[i].s <= 1e-13 * smax) break;
    kept[cand[i].blk].push_back(cand[i].row);        // descending singular value inside the block
    is_kept[i] = 1;
    ++nk;
  }
  double disc = 0.0;
  for (size_t i = cand.size(); i-- > 0;)              // smallest first
    if (!is_kept[i]) disc += cand[i].s * cand[i].s;
  if (discarded_host) *discarded_host = disc;

  // ---- isometries in the boundary layout: sectors of the chosen side ascending, O^T = kept vectors
  std::vector<int> by_sector(nB);
  std::iota(by_sector.begin(), by_sector.end(), 0);
  if (side == HPSI_SIDE_RIGHT)                         // psi blocks are stored by ascending LEFT sector
    std::sort(by_sector.begin(), by_sector.end(), [&](int x, int y) { return sc.blocks[x].right < sc.blocks[y].right; });
  std::vector<IsoRow> rows;
  int64_t dst = 0;
  for (int b : by_sector) {
    const SvdBlk& s = tab[b];
    chi_host[side == HPSI_SIDE_LEFT ? sc.blocks[b].left : sc.blocks[b].right] = (int32_t)kept[b].size();
    for (int row : kept[b]) {
      if (s.tall) rows.push_back({s.w_off + (int64_t)row * s.L, dst, 1.0 / sig[s.row0 + row], s.rows, 0});
      else rows.push_back({s.w_off + (int64_t)row * s.L + s.cols, dst, 1.0, s.rows, 0});
      dst += s.rows;
    }
  }
  if (!rows.empty()) {
    HPSI_CUDA(cudaMemcpyAsync(d_rows, rows.data(), rows.size() * sizeof(IsoRow), cudaMemcpyHostToDevice, st));
    launch_dependent(svd_gather_kernel, dim3(std::min<int>((int)rows.size(), 1024)), dim3(128), 0, st, d_rows, (int)rows.size(), d_w, ot_dev);
    HPSI_CUDA(cudaStreamSynchronize(st));              // `rows` must outlive the copy
  }
  HPSI_CUDA(cudaGetLastError());
  return HPSI_OK;
}

extern "C" int hpsi_truncate(hpsi_plan_t* p, const double* psi_dev, int32_t side, int32_t chi_max, double eps_discard,
                             double* ot_dev, int32_t* chi_host, double* sigma_host, double* discarded_host, void* cuda_stream) {
  return truncate_impl(p, psi_dev, side, chi_max, eps_discard, ot_dev, chi_host, sigma_host, discarded_host, cuda_stream,
                       nullptr, 0);
}

extern "C" int hpsi_truncate_static(hpsi_plan_t* p, const double* psi_dev, int32_t side, int32_t chi_max,
                                    double eps_discard, double* ot_dev, int32_t* chi_host, double* sigma_host,
                                    double* discarded_host, void* cuda_stream) {
  if (!p) { set_error("null plan"); return HPSI_EINVAL; }
  if (p->host_only) { set_error("host-only plan: hpsi_truncate_static needs a CUDA device (no CPU fallback)"); return HPSI_ESTATE; }
  char* scratch = nullptr;
  if (int rc = truncate_static_scratch(&scratch)) return rc;
  return truncate_impl(p, psi_dev, side, chi_max, eps_discard, ot_dev, chi_host, sigma_host, discarded_host, cuda_stream,
                       scratch, sizeof g_truncate_scratch);
}
