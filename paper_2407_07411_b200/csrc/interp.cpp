// Host interpreter of the device schedule (hpsi_debug_interpret): walks exactly the tables the kernels consume
// - prep (padded psi / psi^T), P1 units, P2 units, ordered reduce - with naive loops, so the planner can be
// verified against the oracle on a box without a GPU.  Test infrastructure for the planner; not a compute path:
// hpsi_apply never calls it.
#include <vector>

#include "plan.h"

namespace hpsi {

void interpret_schedule(const Schedule& sc, const double* a, const double* b, const double* psi, double* out, int nvec) {
  std::vector<double> wsv((size_t)sc.ws_len, 0.0);
  double* ws = wsv.data();
  // prep: the copies of vector v sit p_vstride / t_vstride after those of vector v - 1
  for (int v = 0; v < nvec; ++v)
    for (const PsiBlk& B : sc.blocks)
      for (int x = 0; x < B.rows; ++x)
        for (int y = 0; y < B.cols; ++y) {
          double val = psi[(int64_t)v * sc.psi_len + B.off + (int64_t)x * B.cols + y];
          ws[B.p_off + v * B.p_vstride + (int64_t)x * B.ldp + y] = val;
          ws[B.t_off + v * B.t_vstride + (int64_t)y * B.ldt + x] = val;
        }
  // P1: T_t[i, j] = coef_t * sum_k X_t[i,k] Y[j,k] for the unit's tile and terms
  for (const P1Unit& u : sc.p1) {
    if (u.vec >= nvec) continue;
    const Group& g = sc.groups[u.group];
    const double* xbase = (g.order == 1) ? a : b;
    const double* y = ws + g.y1_off + (int64_t)u.vec * g.N1 * g.ldy1;     // vector v: rows [v N1, (v + 1) N1) of the stacked operand
    for (int t = u.t0; t < u.t1; ++t) {
      const Seg& sg = sc.segs[g.seg0 + t];
      // element (i, k) of the operator block: plain storage [i][k], transposed storage [k][i]; the layout is the UNIT's
      // flag, as in the kernels (one layout per unit), not the seg's
      const int64_t xsi = u.xtrans ? 1 : sg.p1_ld, xsk = u.xtrans ? sg.p1_ld : 1;
      for (int r = 0; r < u.rows_valid; ++r) {
        const double* xr = xbase + sg.p1_off + (int64_t)(u.i0 + r) * xsi;
        for (int c = 0; c < u.cols_valid; ++c) {
          const int j = u.j0 + c;
          const double* yr = y + (int64_t)j * g.ldy1;
          double s = 0.0;
          for (int k = 0; k < g.K1; ++k) s += xr[k * xsk] * yr[k];
          ws[g.ws_off + ((int64_t)t * g.rows + u.i0 + r) * g.ldw + u.vec * g.N1p + j] = sg.coef * s;
        }
      }
    }
  }
  // P2: partial[i,j] = sum over runs, segs, k of X[i,k] Y[j,k]
  for (const P2Unit& u : sc.p2) {
    if (u.vec >= nvec) continue;
    for (int r = 0; r < u.rows_valid; ++r)
      for (int c = 0; c < u.cols_valid; ++c) {
        double s = 0.0;
        for (int ri = u.run_begin; ri < u.run_end; ++ri) {
          const Run& run = sc.runs[ri];
          for (int si = run.seg_begin; si < run.seg_end; ++si) {
            const Seg& sg = sc.segs[si];
            const int64_t t_off = run.ws_off + (int64_t)(si - run.seg0) * run.rows * run.ldw + u.vec * run.Kp;
            const int64_t osi = run.trans ? 1 : sg.p2_ld, osk = run.trans ? sg.p2_ld : 1;   // operator block strides: the RUN's layout flag, as in the kernels
            const double *xr, *yr;
            int64_t xsk = 1, ysk = 1;
            if (run.order == 1) {
              xr = ws + t_off + (int64_t)(u.i0 + r) * run.ldw;
              yr = b + sg.p2_off + (int64_t)(u.j0 + c) * osi;
              ysk = osk;
            } else {
              xr = a + sg.p2_off + (int64_t)(u.i0 + r) * osi;
              xsk = osk;
              yr = ws + t_off + (int64_t)(u.j0 + c) * run.ldw;
            }
            for (int k = 0; k < run.K; ++k) s += xr[k * xsk] * yr[k * ysk];
          }
        }
        ws[u.out_off + (int64_t)r * u.ldo + c] = s;
      }
  }
  // fused units: per segment the first GEMM into a local buffer (the kernel's shared-memory operand tile), then the second
  for (const P2Unit& u : sc.pf) {
    std::vector<double> acc((size_t)u.rows_valid * u.cols_valid, 0.0);
    for (int ri = u.run_begin; ri < u.run_end; ++ri) {
      const Run& run = sc.runs[ri];
      const int rows_a = (run.order == 1) ? u.rows_valid : u.cols_valid, row_a0 = (run.order == 1) ? u.i0 : u.j0;
      const double* arena_a = (run.order == 1) ? a : b;
      const double* arena_b = (run.order == 1) ? b : a;
      std::vector<double> c1((size_t)rows_a * run.K);
      for (int si = run.seg_begin; si < run.seg_end; ++si) {
        const Seg& sg = sc.segs[si];
        for (int i = 0; i < rows_a; ++i)
          for (int j = 0; j < run.K; ++j) {
            const double* xr = arena_a + sg.p1_off + (int64_t)(row_a0 + i) * sg.p1_ld;
            const double* yr = ws + run.y1_off + (int64_t)j * run.ldy1;
            double s = 0.0;
            for (int k = 0; k < run.K1; ++k) s += xr[k] * yr[k];
            c1[(size_t)i * run.K + j] = sg.coef * s;
          }
        for (int r = 0; r < u.rows_valid; ++r)
          for (int c = 0; c < u.cols_valid; ++c) {
            double s = 0.0;
            if (run.order == 1) {
              const double* yr = arena_b + sg.p2_off + (int64_t)(u.j0 + c) * sg.p2_ld;
              for (int k = 0; k < run.K; ++k) s += c1[(size_t)r * run.K + k] * yr[k];
            } else {
              const double* xr = arena_b + sg.p2_off + (int64_t)(u.i0 + r) * sg.p2_ld;
              for (int k = 0; k < run.K; ++k) s += xr[k] * c1[(size_t)c * run.K + k];
            }
            acc[(size_t)r * u.cols_valid + c] += s;
          }
      }
    }
    for (int r = 0; r < u.rows_valid; ++r)
      for (int c = 0; c < u.cols_valid; ++c) ws[u.out_off + (int64_t)r * u.ldo + c] = acc[(size_t)r * u.cols_valid + c];
  }
  // ordered reduce (partials: split-major, vector-minor)
  for (int v = 0; v < nvec; ++v)
    for (const PsiBlk& B : sc.blocks)
      for (int x = 0; x < B.rows; ++x)
        for (int y = 0; y < B.cols; ++y) {
          double s = 0.0;
          for (int sp = 0; sp < B.nsplit; ++sp)
            s += ws[B.part_off + ((int64_t)sp * sc.nvec + v) * B.rows * B.ldo + (int64_t)x * B.ldo + y];
          out[(int64_t)v * sc.psi_len + B.off + (int64_t)x * B.cols + y] = s;
        }
}

}  // namespace hpsi
