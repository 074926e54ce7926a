// Renormalised-operator update  A'_t[l,l'] = O_l^T A_t[l,l'] O_l'  (include/hpsi.h "Site update", SURVEY.md 8(f)-4,
// DESIGN.md section 9) on the grouped DMMA engine of hpsi_apply.
//
// Both GEMMs are "NT" launches of the first-GEMM kernel (kernels.cu p1_kernel<TMA, ROT=true>: per-term X operand, one
// shared Y operand per group, the stage ring running across the group's terms, tile stored TRANSPOSED):
//   launch 1, group (l,l'):  X_t = A_t (d_l x d_l'),       Y = O_l'^T (chi_l' x d_l')  ->  T_t^T (chi_l' x d_l)  in the workspace
//   launch 2, group (l,l'):  X_t = T_t^T (chi_l' x d_l),   Y = O_l^T  (chi_l  x d_l )  ->  A'_t  (chi_l  x chi_l') in the output arena
// The contraction order is fixed (right index first: 2 d d' chi' + 2 chi d chi' flops); the other order would need A_t
// as an M-contiguous operand.  The isometries are copied into 32-byte-row padded workspace matrices first (rot_prep).
#include <algorithm>
#include <cstdio>
#include <cstring>
#include <new>
#include <unordered_map>

#include "plan_dev.h"

namespace hpsi {

struct IsoCopy {              // O_l^T: dense chi x d at src_off of the caller's array -> padded chi x ld at dst_off of the workspace
  int64_t src_off, dst_off;
  int32_t rows, cols, ld, pad;
};

__global__ void rot_prep_kernel(const IsoCopy* iso, const double* __restrict__ ot, double* __restrict__ ws) {
  pdl_wait();
  const IsoCopy c = iso[blockIdx.y];
  const int n = c.rows * c.cols;
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
    const int a = e / c.cols, x = e - a * c.cols;
    ws[c.dst_off + (int64_t)a * c.ld + x] = ot[c.src_off + e];
  }
}

}  // namespace hpsi

using namespace hpsi;

struct hpsi_rotate {
  struct hpsi_plan core;                       // schedule tables (groups / segs / p1 units of both launches), workspace, tensor maps
  int n_units1 = 0, n_units2 = 0;
  std::vector<IsoCopy> iso;
  IsoCopy* d_iso = nullptr;
  int max_iso_elems = 0;
  std::vector<hpsi_opblock_t> out_blocks;
  int64_t out_len = 0, iso_len = 0, useful_flops = 0, algo_bytes = 0, inter_bytes = 0;
};

namespace {

int64_t align4(int64_t x) { return (x + 3) & ~(int64_t)3; }

#define RFAIL(code, ...)                                  \
  do {                                                    \
    char buf_[512];                                       \
    snprintf(buf_, sizeof buf_, __VA_ARGS__);             \
    set_error(buf_);                                      \
    return code;                                          \
  } while (0)

// P1-style units of one group: tile positions of the (rows x N1) product, ranges of ~stages_per_unit K-tiles of terms
void add_units(Schedule& sc, int gi, int stages_per_unit) {
  const Group& g = sc.groups[gi];
  const int stages = (g.K1 + KT - 1) / KT;
  if (g.N1p > 0) {                                   // stacked second launch: "terms" are 64-row slabs, a unit = a range of slabs
    const int nslab = (g.rows + TILE - 1) / TILE;
    int ns = std::max(1, std::min(nslab, (stages_per_unit + stages - 1) / stages));
    const int nchunk = (nslab + ns - 1) / ns;
    ns = (nslab + nchunk - 1) / nchunk;
    auto ct = split_cols(g.N1);
    const int rows_first = std::min(g.rows, TILE);
    for (int t0 = 0; t0 < nslab; t0 += ns) {
      const int t1 = std::min(nslab, t0 + ns);
      for (auto& c : ct) {
        const int32_t grid = best_grid(frags(rows_first), frags(c.len));
        sc.p1.push_back({gi, t0, t1, 0, rows_first, c.start, c.len, grid, 0, 0});
        sc.issued_flops += (int64_t)frags(rows_first) * frags(c.len) * ((g.K1 + 3) / 4) * 512 * (t1 - t0);
      }
    }
    return;
  }
  int nt = std::max(1, std::min(g.tcount, (stages_per_unit + stages - 1) / stages));
  const int nchunk = (g.tcount + nt - 1) / nt;
  nt = (g.tcount + nchunk - 1) / nchunk;
  auto rt = split_rows(g.rows);
  auto ct = split_cols(g.N1);
  for (int t0 = 0; t0 < g.tcount; t0 += nt) {
    const int t1 = std::min(g.tcount, t0 + nt);
    for (auto& r : rt)
      for (auto& c : ct) {
        const int32_t grid = best_grid(frags(r.len), frags(c.len));
        sc.p1.push_back({gi, t0, t1, r.start, r.len, c.start, c.len, grid, 0, 0});
        sc.issued_flops += (int64_t)frags(r.len) * frags(c.len) * ((g.K1 + 3) / 4) * 512 * (t1 - t0);
      }
  }
}

int build_rotate(hpsi_rotate* r, int32_t nsec, const int32_t* d, const int32_t* chi, int64_t nb, const hpsi_opblock_t* blk,
                 int64_t a_len, int n_sm) {
  Schedule& sc = r->core.sc;
  if (nsec < 0 || nb < 0) RFAIL(HPSI_EINVAL, "negative sector / block count");
  if ((nsec > 0 && (!d || !chi)) || (nb > 0 && !blk)) RFAIL(HPSI_EINVAL, "null argument");
  for (int l = 0; l < nsec; ++l) {
    if (d[l] < 1) RFAIL(HPSI_EINVAL, "sector %d has dimension %d < 1", l, d[l]);
    if (chi[l] < 0 || chi[l] > d[l]) RFAIL(HPSI_EINVAL, "sector %d: kept dimension %d outside 0..%d", l, chi[l], d[l]);
  }
  sc.aligned16 = true;
  std::unordered_map<uint64_t, int64_t> seen;
  for (int64_t i = 0; i < nb; ++i) {
    const hpsi_opblock_t& e = blk[i];
    if (e.row < 0 || e.row >= nsec || e.col < 0 || e.col >= nsec) RFAIL(HPSI_EINVAL, "block %lld: sector index out of range", (long long)i);
    if (e.term < 0) RFAIL(HPSI_EINVAL, "block %lld: negative term", (long long)i);
    if (e.ld < d[e.col]) RFAIL(HPSI_EINVAL, "block %lld: ld %d < cols %d", (long long)i, e.ld, d[e.col]);
    if (e.offset < 0) RFAIL(HPSI_EINVAL, "block %lld: negative offset", (long long)i);
    const int64_t last = e.offset + (int64_t)(d[e.row] - 1) * e.ld + d[e.col];
    if (a_len > 0 && last > a_len) RFAIL(HPSI_EINVAL, "block %lld: extends past the arena", (long long)i);
    const uint64_t key = ((uint64_t)e.term * (uint64_t)nsec + (uint64_t)e.row) * (uint64_t)nsec + (uint64_t)e.col;
    if (!seen.emplace(key, i).second) RFAIL(HPSI_EINVAL, "two blocks for (term %d, row %d, col %d)", e.term, e.row, e.col);
  }

  // ---- isometries: boundary layout -> padded workspace copies, one tensor map each
  int64_t ws = 0, src = 0;
  std::vector<int64_t> iso_off(nsec, -1);
  std::vector<int32_t> iso_ld(nsec, 0), iso_map(nsec, -1);
  auto add_map = [&](int base, int64_t moff, int rows, int cols, int ld) -> int32_t {
    sc.maps.push_back({moff, base, rows, cols, ld, TILE, KT});
    return (int32_t)sc.maps.size() - 1;
  };
  for (int l = 0; l < nsec; ++l) {
    if (chi[l] > 0) {
      iso_ld[l] = sector_up(d[l]);
      iso_off[l] = ws;
      iso_map[l] = add_map(BASE_WS, ws, chi[l], d[l], iso_ld[l]);
      r->iso.push_back({src, ws, chi[l], d[l], iso_ld[l], 0});
      r->max_iso_elems = std::max(r->max_iso_elems, chi[l] * d[l]);
      ws = (ws + (int64_t)chi[l] * iso_ld[l] + 15) & ~(int64_t)15;
    }
    src += (int64_t)chi[l] * d[l];
  }
  r->iso_len = src;

  // ---- output layout (input order) and the surviving blocks sorted into (l, l') groups
  r->out_blocks.assign(blk, blk + nb);
  std::vector<int64_t> alive;
  int64_t out = 0;
  for (int64_t i = 0; i < nb; ++i) {
    hpsi_opblock_t& o = r->out_blocks[i];
    if (chi[o.row] == 0 || chi[o.col] == 0) { o.ld = 0; o.offset = -1; continue; }
    o.ld = sector_up(chi[o.col]);
    o.offset = out;
    out = align4(out + (int64_t)chi[o.row] * o.ld);
    alive.push_back(i);
    const int64_t dl = d[o.row], dc = d[o.col], cl = chi[o.row], cc = chi[o.col];
    r->useful_flops += 2 * dl * dc * cc + 2 * cl * dl * cc;
    r->algo_bytes += 8 * (dl * dc + cl * cc);
    r->inter_bytes += 8 * cc * dl;
    if ((blk[i].offset & 1) || (blk[i].ld & 1)) sc.aligned16 = false;
  }
  r->out_len = std::max<int64_t>(out, 4);
  std::stable_sort(alive.begin(), alive.end(), [&](int64_t x, int64_t y) {
    if (blk[x].row != blk[y].row) return blk[x].row < blk[y].row;
    return blk[x].col < blk[y].col;
  });

  // ---- groups and segs of launch 1, then of launch 2 (same (l,l') groups, same order of blocks)
  auto group_end = [&](size_t i) {                     // one past the last block of the (row, col) group starting at i
    size_t j = i;
    while (j < alive.size() && blk[alive[j]].row == blk[alive[i]].row && blk[alive[j]].col == blk[alive[i]].col) ++j;
    return j;
  };
  sc.segs.reserve(2 * alive.size());
  std::vector<int64_t> tt_off(alive.size());          // workspace offset of T_t^T, in `alive` order
  for (size_t i = 0; i < alive.size();) {
    const size_t j = group_end(i);
    const int l = blk[alive[i]].row, lp = blk[alive[i]].col;
    Group g{};
    g.order = 1;                          // X operands come from the A arena (DevSchedule.a)
    g.tcount = (int32_t)(j - i);
    g.seg0 = (int32_t)sc.segs.size();
    g.rows = d[l]; g.K1 = d[lp]; g.N1 = chi[lp];
    g.ldw = sector_up(d[l]);              // leading dimension of T_t^T (chi_l' x d_l)
    g.ldy1 = iso_ld[lp]; g.y1_off = iso_off[lp]; g.y1_map = iso_map[lp];
    g.ws_off = ws;
    g.ws_map = -1;
    g.src = lp; g.dst = l;
    // The T_t^T of a group sit one under the other, sector_up(chi_l') rows each (the pad rows stay zero: the workspace is
    // zeroed at plan time and never written there), so that the second launch can read them as ONE stacked matrix.
    const int chip = sector_up(chi[lp]);
    for (size_t q = i; q < j; ++q) {
      const hpsi_opblock_t& e = blk[alive[q]];
      Seg sg{};
      sg.p1_off = e.offset; sg.p1_ld = e.ld;
      sg.p1_map = add_map(BASE_A, e.offset, d[l], d[lp], e.ld);
      sg.p2_off = ws; sg.p2_ld = g.ldw;   // where the transposed tile of this term goes
      sg.p2_map = -1;
      sg.coef = 1.0;
      tt_off[q] = ws;
      ws += (int64_t)chip * g.ldw;
      sc.segs.push_back(sg);
    }
    ws = (ws + 15) & ~(int64_t)15;
    sc.groups.push_back(g);
    i = j;
  }
  const int ng1 = (int)sc.groups.size();
  for (size_t i = 0; i < alive.size();) {
    const size_t j = group_end(i);
    const int l = blk[alive[i]].row, lp = blk[alive[i]].col;
    // Second launch, STACKED: the group's T_t^T form one matrix of tcount x chip rows (chip = sector_up(chi_l') per block,
    // chi_l' of them real); a CTA works on 64-row slabs of it - 2 to 3 blocks at once instead of one chi' x chi tile
    // (~25 x 25, a quarter of a CTA tile) per block - and scatters every row to its block's A' (kernels.cu p1_consume).
    const int chip = sector_up(chi[lp]);
    Group g{};
    g.order = 2;                          // X operands come from DevSchedule.b, which the update points at the workspace
    g.tcount = (int32_t)(j - i);
    g.seg0 = (int32_t)sc.segs.size();
    g.rows = g.tcount * chip;             // rows of the stacked matrix
    g.K1 = d[l]; g.N1 = chi[l];
    g.N1p = chip;                         // > 0 marks the stacked mode: rows per block ...
    g.ldw = chi[lp];                      // ... of which this many are real
    g.ldy1 = iso_ld[l]; g.y1_off = iso_off[l]; g.y1_map = iso_map[l];
    g.ws_off = 0; g.ws_map = -1;
    g.src = lp; g.dst = l;
    const int ldt = sector_up(d[l]);
    const int32_t stack_map = add_map(BASE_WS, tt_off[i], g.rows, d[l], ldt);
    for (size_t q = i; q < j; ++q) {
      const hpsi_opblock_t& o = r->out_blocks[alive[q]];
      Seg sg{};
      sg.p1_off = tt_off[i]; sg.p1_ld = ldt;            // the stacked matrix (every seg: the kernel reads seg0's)
      sg.p1_map = stack_map;
      sg.p2_off = o.offset; sg.p2_ld = o.ld;
      sg.p2_map = -1;
      sg.coef = 1.0;
      sc.segs.push_back(sg);
    }
    sc.groups.push_back(g);
    i = j;
  }

  // ---- units: ~96 K-tiles per CTA, fewer when the launch would otherwise be only a few waves
  sc.issued_flops = 0;
  for (int launch = 0; launch < 2; ++launch) {
    const int g0 = launch ? ng1 : 0, g1 = launch ? (int)sc.groups.size() : ng1;
    int64_t total = 0;
    for (int gi = g0; gi < g1; ++gi) {
      const Group& g = sc.groups[gi];
      total += (g.N1p > 0 ? (int64_t)((g.rows + TILE - 1) / TILE) * split_cols(g.N1).size()
                          : (int64_t)split_rows(g.rows).size() * split_cols(g.N1).size() * g.tcount) * ((g.K1 + KT - 1) / KT);
    }
    const int spu = (int)std::max<int64_t>(12, std::min<int64_t>(96, total / ((int64_t)std::max(n_sm, 1) * 3 * 8)));
    // heaviest groups first
    std::vector<int> order;
    for (int gi = g0; gi < g1; ++gi) order.push_back(gi);
    std::stable_sort(order.begin(), order.end(), [&](int x, int y) {
      const Group &a = sc.groups[x], &b = sc.groups[y];
      const int64_t ca = (int64_t)std::min(frags(a.rows), TILE_M / 8) * std::min(frags(a.N1), TILE / 8) * a.K1;
      const int64_t cb = (int64_t)std::min(frags(b.rows), TILE_M / 8) * std::min(frags(b.N1), TILE / 8) * b.K1;
      return ca > cb;
    });
    const size_t before = sc.p1.size();
    for (int gi : order) add_units(sc, gi, spu);
    (launch ? r->n_units2 : r->n_units1) = (int)(sc.p1.size() - before);
  }
  sc.useful_flops = r->useful_flops;
  sc.ws_len = std::max<int64_t>(ws, 16);
  return HPSI_OK;
}

void free_rotate(hpsi_rotate* r) {
  if (!r) return;
  if (r->core.device_ok) {
    cudaFree(r->d_iso);
    cudaFree(r->core.d_tables);
    cudaFree(r->core.d_ws);
    cudaFree(r->core.d_maps);
    cudaGetLastError();
  }
  delete r;
}

}  // namespace

extern "C" int hpsi_rotate_plan(int32_t n_sectors, const int32_t* d, const int32_t* chi, int64_t n_blocks,
                                const hpsi_opblock_t* blocks, const double* a_data_dev, int64_t a_len, uint32_t flags,
                                hpsi_rotate_t** out) {
  if (!out) { set_error("null out"); return HPSI_EINVAL; }
  *out = nullptr;
  hpsi_rotate* r = new (std::nothrow) hpsi_rotate();
  if (!r) { set_error("out of host memory"); return HPSI_ENOMEM; }
  struct hpsi_plan& p = r->core;
  p.host_only = (flags & HPSI_PLAN_HOST_ONLY) != 0;
  int rc = HPSI_OK;
  try {
    if (!p.host_only) {
      int dev = 0;
      cudaError_t e = cudaGetDevice(&dev);
      if (e == cudaSuccess) e = cudaDeviceGetAttribute(&p.n_sm, cudaDevAttrMultiProcessorCount, dev);
      if (e == cudaSuccess) e = kernels_init();
      if (e != cudaSuccess) {
        rc = cuda_fail(e, "device initialisation (no CPU fallback exists)");
        free_rotate(r);
        return rc;
      }
      p.device_ok = true;
    }
    rc = build_rotate(r, n_sectors, d, chi, n_blocks, blocks, a_len, p.n_sm);
    if (rc != HPSI_OK) { free_rotate(r); return rc; }
    if (!p.host_only) {
      if (!r->core.sc.segs.empty() && !a_data_dev) { set_error("null operator arena"); free_rotate(r); return HPSI_EINVAL; }
      rc = upload_schedule(&p);
      if (rc != HPSI_OK) { free_rotate(r); return rc; }
      if (!r->iso.empty()) {
        cudaError_t e = cudaMalloc(&r->d_iso, r->iso.size() * sizeof(IsoCopy));
        if (e == cudaSuccess) e = cudaMemcpy(r->d_iso, r->iso.data(), r->iso.size() * sizeof(IsoCopy), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) { rc = cuda_fail(e, "isometry table upload"); free_rotate(r); return rc; }
      }
      p.dev.a = a_data_dev;
      p.dev.b = p.d_ws;                 // launch 2 reads its per-term operand (T_t^T) through the "B arena" pointer
      p.dev.n_blocks = 0;
      p.dev.paired = 0;
      p.aligned16 = p.sc.aligned16 && ((reinterpret_cast<uintptr_t>(a_data_dev) & 15) == 0);
      if (p.aligned16) {
        rc = encode_maps(&p);
        if (rc != HPSI_OK) { free_rotate(r); return rc; }
      }
      p.bound = true;
    }
  } catch (const std::bad_alloc&) {
    set_error("out of host memory while planning");
    free_rotate(r);
    return HPSI_ENOMEM;
  }
  *out = r;
  return HPSI_OK;
}

static int rotate_launch(hpsi_rotate* r, const double* ot_dev, double* out_dev, cudaStream_t st, cudaEvent_t* ev) {
  struct hpsi_plan& p = r->core;
  if (ev) HPSI_CUDA(cudaEventRecord(ev[0], st));
  if (!r->iso.empty()) {
    int gx = std::min(64, std::max(1, (r->max_iso_elems + 255) / 256));
    launch_dependent(rot_prep_kernel, dim3(dim3(gx, (unsigned)r->iso.size())), dim3(256), 0, st, r->d_iso, ot_dev, p.d_ws);
  }
  if (ev) HPSI_CUDA(cudaEventRecord(ev[1], st));
  DevSchedule d1 = p.dev;
  d1.n_p1 = r->n_units1;
  d1.rot_dst = p.d_ws;
  launch_p1_rot(d1, p.aligned16, st);
  if (ev) HPSI_CUDA(cudaEventRecord(ev[2], st));
  DevSchedule d2 = p.dev;
  d2.p1 = p.dev.p1 + r->n_units1;
  d2.n_p1 = r->n_units2;
  d2.rot_dst = out_dev;
  launch_p1_rot(d2, p.aligned16, st);
  if (ev) HPSI_CUDA(cudaEventRecord(ev[3], st));
  HPSI_CUDA(cudaGetLastError());
  return HPSI_OK;
}

static int rotate_check(hpsi_rotate* r, const double* ot_dev, double* out_dev) {
  if (!r) { set_error("null object"); return HPSI_EINVAL; }
  if (r->core.host_only) { set_error("host-only object: hpsi_rotate_apply needs a CUDA device (no CPU fallback)"); return HPSI_ESTATE; }
  if (r->core.sc.segs.empty()) return 1;            // nothing survives: nothing to do
  if (!ot_dev || !out_dev) { set_error("null isometries / output"); return HPSI_EINVAL; }
  return HPSI_OK;
}

extern "C" int hpsi_rotate_apply(hpsi_rotate_t* r, const double* ot_dev, double* out_dev, void* cuda_stream) {
  const int rc = rotate_check(r, ot_dev, out_dev);
  if (rc != HPSI_OK) return rc > 0 ? HPSI_OK : rc;
  return rotate_launch(r, ot_dev, out_dev, static_cast<cudaStream_t>(cuda_stream), nullptr);
}

extern "C" int hpsi_rotate_apply_profiled(hpsi_rotate_t* r, const double* ot_dev, double* out_dev, void* cuda_stream,
                                          float* ms_host) {
  if (!ms_host) { set_error("null ms_host"); return HPSI_EINVAL; }
  ms_host[0] = ms_host[1] = ms_host[2] = 0.f;
  const int rc = rotate_check(r, ot_dev, out_dev);
  if (rc != HPSI_OK) return rc > 0 ? HPSI_OK : rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  EventSet<4> ev;
  HPSI_CUDA(ev.create());
  int rc2 = rotate_launch(r, ot_dev, out_dev, st, ev.ev);
  if (rc2 == HPSI_OK) {
    HPSI_CUDA(cudaEventSynchronize(ev[3]));
    for (int i = 0; i < 3; ++i) HPSI_CUDA(cudaEventElapsedTime(&ms_host[i], ev[i], ev[i + 1]));
  }
  return rc2;
}

extern "C" int hpsi_rotate_query(const hpsi_rotate_t* r, int what, void* out, size_t bytes) {
  if (!r || !out) { set_error("null argument"); return HPSI_EINVAL; }
  auto put = [&](int64_t v) -> int {
    if (bytes < sizeof v) { set_error("hpsi_rotate_query: buffer too small"); return HPSI_EINVAL; }
    memcpy(out, &v, sizeof v);
    return HPSI_OK;
  };
  switch (what) {
    case HPSI_RQ_OUT_LENGTH: return put(r->out_len);
    case HPSI_RQ_OUT_BLOCKS:
      if (bytes < r->out_blocks.size() * sizeof(hpsi_opblock_t)) { set_error("hpsi_rotate_query: buffer too small"); return HPSI_EINVAL; }
      if (!r->out_blocks.empty()) memcpy(out, r->out_blocks.data(), r->out_blocks.size() * sizeof(hpsi_opblock_t));
      return HPSI_OK;
    case HPSI_RQ_ISO_LENGTH: return put(r->iso_len);
    case HPSI_RQ_USEFUL_FLOPS: return put(r->useful_flops);
    case HPSI_RQ_ALGO_BYTES: return put(r->algo_bytes);
    case HPSI_RQ_WORKSPACE_BYTES: return put(r->core.sc.ws_len * 8);
    case HPSI_RQ_N_UNITS_1: return put(r->n_units1);
    case HPSI_RQ_N_UNITS_2: return put(r->n_units2);
    case HPSI_RQ_ALIGNED16: return put(r->core.host_only ? r->core.sc.aligned16 : r->core.aligned16);
    case HPSI_RQ_INTERMEDIATE_BYTES: return put(r->inter_bytes);
    default: set_error("hpsi_rotate_query: unknown item"); return HPSI_EINVAL;
  }
}

extern "C" void hpsi_rotate_destroy(hpsi_rotate_t* r) { free_rotate(r); }

// Host walk of the device tables (tests only): isometry copies, then the units of both launches with naive loops.
extern "C" int hpsi_rotate_debug_interpret(const hpsi_rotate_t* r, const double* a_host, const double* ot_host, double* out_host) {
  if (!r) { set_error("null object"); return HPSI_EINVAL; }
  const Schedule& sc = r->core.sc;
  if (sc.segs.empty()) return HPSI_OK;
  if (!a_host || !ot_host || !out_host) { set_error("null argument"); return HPSI_EINVAL; }
  try {
    std::vector<double> wsv((size_t)sc.ws_len, 0.0);
    double* ws = wsv.data();
    for (const IsoCopy& c : r->iso)
      for (int a = 0; a < c.rows; ++a)
        for (int x = 0; x < c.cols; ++x) ws[c.dst_off + (int64_t)a * c.ld + x] = ot_host[c.src_off + (int64_t)a * c.cols + x];
    for (size_t ui = 0; ui < sc.p1.size(); ++ui) {
      const P1Unit& u = sc.p1[ui];
      const bool second = (int)ui >= r->n_units1;
      const Group& g = sc.groups[u.group];
      const double* xbase = (g.order == 1) ? a_host : ws;
      double* dst = second ? out_host : ws;
      for (int t = u.t0; t < u.t1; ++t) {
        if (g.N1p > 0) {                       // stacked second launch: slab t of the stacked T^T, rows scattered to their blocks
          const Seg& s0 = sc.segs[g.seg0];
          for (int i = 0; i < TILE; ++i) {
            const int R = t * TILE + i;
            if (R >= g.rows) break;
            const int b = R / g.N1p, a = R - b * g.N1p;
            if (a >= g.ldw) continue;
            const Seg& sg = sc.segs[g.seg0 + b];
            for (int j = 0; j < u.cols_valid; ++j) {
              const double* xr = xbase + s0.p1_off + (int64_t)R * s0.p1_ld;
              const double* yr = ws + g.y1_off + (int64_t)(u.j0 + j) * g.ldy1;
              double s = 0.0;
              for (int k = 0; k < g.K1; ++k) s += xr[k] * yr[k];
              dst[sg.p2_off + (int64_t)(u.j0 + j) * sg.p2_ld + a] = s;
            }
          }
          continue;
        }
        const Seg& sg = sc.segs[g.seg0 + t];
        for (int i = 0; i < u.rows_valid; ++i)
          for (int j = 0; j < u.cols_valid; ++j) {
            const double* xr = xbase + sg.p1_off + (int64_t)(u.i0 + i) * sg.p1_ld;
            const double* yr = ws + g.y1_off + (int64_t)(u.j0 + j) * g.ldy1;
            double s = 0.0;
            for (int k = 0; k < g.K1; ++k) s += xr[k] * yr[k];
            dst[sg.p2_off + (int64_t)(u.j0 + j) * sg.p2_ld + u.i0 + i] = s;
          }
      }
    }
  } catch (const std::bad_alloc&) {
    set_error("out of host memory in interpreter");
    return HPSI_ENOMEM;
  }
  return HPSI_OK;
}
